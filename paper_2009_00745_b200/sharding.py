"""State sharding for multi-GPU runs (one process per GPU).

The quasiparticle states are independent between the two density barriers of a time step
("each GPU ... nwfip wavefunctions", partial densities summed with
MPI_Allreduce).  Each rank owns a contiguous range of the states of each species with all their
multistep history; grid fields (densities, potentials) are replicated.  The one collective is an
in-place all-reduce (sum) of the 2 x 13 x Nxyz density accumulators at each barrier, issued on
device buffers through the library's reduce hook (NCCL over NVLink on the GPU box).
This module holds host logic only: no arithmetic of the method.
"""
import torch
import torch.distributed as dist


def shard_range(nwf, world, rank):
    """[first, last) of the states rank `rank` owns: contiguous, sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world) or nwf < 0:
        raise ValueError((nwf, world, rank))
    base, extra = divmod(nwf, world)
    first = rank * base + min(rank, extra)
    return first, first + base + (1 if rank < extra else 0)


def shard_counts(nwf, world):
    return [shard_range(nwf, world, r)[1] - shard_range(nwf, world, r)[0] for r in range(world)]


def allreduce_sum_(t, group=None):
    """in-place sum over ranks (no-op without an initialised process group)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t


def _allreduce_ints(vals, op, group=None):
    """element-wise reduction over ranks of a few host integers (identity without an initialised process group)."""
    if not (dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1):
        return list(vals)
    t = torch.tensor(list(vals), dtype=torch.int64)
    if dist.get_backend(group) == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=op, group=group)
    return [int(v) for v in t.cpu()]


def attach(ctx, group=None, global_nwf=None, coulomb=None):
    """make `ctx` (paper_2009_00745_b200.lise.Lise) sum its density accumulators over the ranks of `group`.
    Coulomb must be the same on every rank (lise.h: the flag alone decides), so it is decided here from what the caller
    asked for and from the GLOBAL proton count: on iff requested and some rank holds proton states.  A rank that
    happens to own no proton state (whose context therefore defaulted to Coulomb off) then still computes the same
    potentials and energy as the others.  The request is ctx.coulomb_requested -- the flag of the params the context
    was given, the library default otherwise; `coulomb` (True / False) overrides it, None keeps it.  The global proton
    count is global_nwf[1] if given, else the sum over ranks of ctx.nwf[1].  Collective: every rank of `group` calls it."""
    if global_nwf is not None:
        global_p = int(global_nwf[1])
    else:
        global_p = _allreduce_ints([ctx.nwf[1]], dist.ReduceOp.SUM, group)[0]
    req = int(bool(ctx.coulomb_requested if coulomb is None else coulomb))
    lo, hi = _allreduce_ints([req, -req], dist.ReduceOp.MIN, group)
    if lo != -hi:
        raise ValueError("sharding.attach: the ranks disagree about Coulomb (params.coulomb must be the same on every rank)")
    want = 1 if (req and global_p > 0) else 0
    if ctx.params.coulomb != want:
        ctx.params.coulomb = want
        ctx.set_params(ctx.params)
        ctx.coulomb_requested = req          # set_params recorded the decided flag; keep the caller's request
    ctx.set_reduce_hook(lambda t: allreduce_sum_(t, group))


def global_observables(obs, group=None):
    """combine per-rank observables: energies and particle numbers come from the (already global)
    densities and are identical on every rank; the defects are maxima over each rank's own states."""
    out = dict(obs)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        t = torch.tensor([obs["norm_defect"], obs["ortho_defect"]], dtype=torch.float64)
        if dist.get_backend(group) == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
        out["norm_defect"], out["ortho_defect"] = float(t[0]), float(t[1])
    return out
