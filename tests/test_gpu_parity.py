"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's north_star:
  wavefunctions <= 1e-10 (max |diff| / max |ref|) after 10 steps, densities <= 1e-11, energy <= 1e-10.
"""
import numpy as np
import pytest
import torch

from oracle import ref
from paper_2009_00745_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_WF, TOL_DENS, TOL_E = 1e-10, 1e-11, 1e-10


def rel(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def field_rel(got, want):
    """per-field max-norm relative error for [nfields, ...] arrays, each field on its OWN scale.  Only a field that is
    zero in the reference -- identically, or to the oracle's own round-off (<= 1e-12 of the largest field: e.g. the
    Laplacian of a constant effective mass, a sum of cancelling terms) -- is compared on the scale of the largest field.
    A field that carries a signal between 1e-12 and 1e-9 of the array scale cannot be compared at the parity tolerance
    on either scale (round-off of the large fields leaks into it): that is a flaw of the test input, and it fails here
    instead of passing unnoticed."""
    scale = np.abs(want).max()
    out = []
    for f in range(want.shape[0]):
        s = np.abs(want[f]).max()
        if s <= 1e-12 * scale:
            out.append(np.abs(got[f] - want[f]).max() / scale if scale > 0.0 else np.abs(got[f]).max())
            continue
        assert s > 1e-9 * scale, (f"field_rel: row {f} has max {s:.3e}, between 1e-12 and 1e-9 of the array scale {scale:.3e}: "
                                  f"too small to compare; error on its own scale {np.abs(got[f] - want[f]).max() / s:.3e}")
        out.append(np.abs(got[f] - want[f]).max() / s)
    return max(out)


CASES = {
    # name: (config index, shape override, dx override, (nwf_n, nwf_p), steps, launch options)
    "config0": (0, None, None, (128, 0), 10, None),            # BASELINE configs[0] in full
    "both_12x8x16": (0, (12, 8, 16), 1.5, (20, 12), 10, None), # non-cubic, both species, Coulomb, ragged chunks
    "r2_6x10x12": (0, (6, 10, 12), 1.5, (7, 5), 6, None),      # sizes not divisible by 4 (R = 2 blocking)
    # 10 steps (3 starter + 7 ABM) on reduced-state versions of configs 1-4; 256 + 256 states on the
    # config-1 lattice in three chunks per species (96 + 96 + 64) with the stream overlap on: the launch configuration
    # bench.py times (full state groups in every CTA, double-buffered W, densities per group of 2 chunks)
    "c1_24c_256": (1, None, None, (256, 256), 10, dict(chunk=96, dgroup=2, overlap=True)),
    # the multi-chunk pipeline: 7 + 4 chunks with ragged tails, double-buffered W / eta, update on the second stream,
    # density launches per group of 3 chunks (a species change inside a group)
    "c1_24c_pipeline": (1, None, None, (40, 24), 10, dict(chunk=6, dgroup=3, overlap=True)),
    # configs 2-4 in the schedule bench.py times as well: three chunks per species with a ragged tail (96 + 96 + 64,
    # 48 + 48 + 32), double-buffered W, update on the second stream, densities per group of 2 chunks.  32^3 (a target
    # workload) at SURVEY 8(c)'s 256 + 256 states; the two long-line lattices at 128 + 128, because the oracle's share of
    # these three cases (about 7 minutes on the box's 16 cores) has to fit the 20 minutes the whole GPU suite is given
    "c2_32c": (2, None, None, (256, 256), 10, dict(chunk=96, dgroup=2, overlap=True)),
    "c3_24x24x64": (3, None, None, (128, 128), 10, dict(chunk=48, dgroup=2, overlap=True)),
    "c4_40c": (4, None, None, (128, 128), 10, dict(chunk=48, dgroup=2, overlap=True)),
    # the paper's own fission box 24^2 x 48 (L1076): 48-point lines = 8 x 6, the size-6 real DFT of the DMMA line operator
    "p_24x24x48": (3, (24, 24, 48), None, (12, 8), 5, None),
}


def make_case(name):
    from paper_2009_00745_b200 import lise
    idx, shape, dx, nwf, steps, opts = CASES[name]
    cfg = dict(inputs.CONFIGS[idx])
    if shape is not None:
        cfg["shape"] = shape
    if dx is not None:
        cfg["dx"] = dx
    psi = [inputs.make_species(cfg, q, nwf[q], seed=inputs.SEED0 + idx) for q in (0, 1)]
    oc = ref.RefContext(*cfg["shape"], cfg["dx"], cfg["dt"], nwf[0], nwf[1])
    gc = lise.Lise(*cfg["shape"], cfg["dx"], cfg["dt"], nwf[0], nwf[1])
    if opts:
        gc.set_chunk(opts["chunk"]); gc.set_density_group(opts["dgroup"]); gc.set_overlap(opts["overlap"])
    for q in (0, 1):
        oc.set_wavefunctions(q, psi[q].numpy())
        gc.set_wavefunctions(q, psi[q].cuda())
    return cfg, psi, oc, gc, steps


@pytest.fixture(scope="module", params=list(CASES))
def case(request):
    c = make_case(request.param)
    yield (request.param,) + c
    c[3].close(); c[2].close()


def test_initial_densities_potentials_and_hpsi(case):
    name, cfg, psi, oc, gc, steps = case
    for q in (0, 1):
        if oc.nwf[q] == 0:
            continue
        d_ref = oc.densities(q); d_gpu = gc.densities(q).cpu().numpy()
        assert field_rel(d_gpu, d_ref) < TOL_DENS, (name, "densities", q)
        p_ref = oc.potentials(q); p_gpu = gc.potentials(q).cpu().numpy()
        assert field_rel(p_gpu, p_ref) < 1e-10, (name, "potentials", q)
        h_ref = oc.apply_h(q, psi[q].numpy()).reshape(psi[q].shape)
        h_gpu = gc.apply_h(q, psi[q].cuda()).cpu().numpy()
        assert rel(h_gpu, h_ref) < 1e-12, (name, "H psi", q)
    o_ref = oc.observables(); o_gpu = gc.observables()
    assert abs(o_gpu["energy"] - o_ref["energy"]) < TOL_E * abs(o_ref["energy"])
    for k in ("e_kin", "e_skyrme", "e_coul", "e_pair", "n_neutron", "n_proton"):
        assert abs(o_gpu[k] - o_ref[k]) < TOL_E * max(abs(o_ref[k]), abs(o_ref["energy"])), (name, k)
    assert o_gpu["norm_defect"] < 1e-12 and o_gpu["ortho_defect"] < 1e-12


def test_time_steps_match_oracle(case):
    name, cfg, psi, oc, gc, steps = case
    oc.step(steps); gc.step(steps)
    for q in (0, 1):
        if oc.nwf[q] == 0:
            continue
        w_ref = oc.get_wavefunctions(q); w_gpu = gc.get_wavefunctions(q).cpu().numpy()
        assert rel(w_gpu, w_ref) < TOL_WF, (name, "wavefunctions", q)
        assert field_rel(gc.densities(q).cpu().numpy(), oc.densities(q)) < TOL_DENS, (name, "densities", q)
    o_ref = oc.observables(); o_gpu = gc.observables()
    assert abs(o_gpu["energy"] - o_ref["energy"]) < TOL_E * abs(o_ref["energy"]), (name, o_gpu, o_ref)
    assert abs(o_gpu["n_neutron"] - o_ref["n_neutron"]) < TOL_E * max(o_ref["n_neutron"], 1.0)
    assert abs(o_gpu["norm_defect"] - o_ref["norm_defect"]) < 1e-12
    assert abs(o_gpu["ortho_defect"] - o_ref["ortho_defect"]) < 1e-12
    assert o_gpu["step"] == steps and abs(o_gpu["time"] - steps * cfg["dt"]) < 1e-12


def test_chunk_size_does_not_change_results():
    """the state-chunking of the launches is an implementation detail: results are bit-identical
    for states (each state's arithmetic is independent) and equal to round-off for densities."""
    from paper_2009_00745_b200 import lise
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (12, 12, 12)
    psi = inputs.make_species(cfg, 0, 37, seed=5).cuda()
    res = []
    for chunk in (0, 5, 37):
        g = lise.Lise(*cfg["shape"], cfg["dx"], 0.05, 37, 0)
        g.set_chunk(chunk)
        g.set_wavefunctions(0, psi)
        g.step(5)
        res.append((g.get_wavefunctions(0).cpu().numpy(), g.densities(0).cpu().numpy()))
        g.close()
    for w, d in res[1:]:
        assert rel(w, res[0][0]) < 1e-13
        assert rel(d, res[0][1]) < 1e-13


@pytest.mark.parametrize("idx", [1, 2, 3, 4])
def test_full_size_single_evaluation_in_the_bench_launch_configuration(idx):
    """BASELINE.json configs[1..4] at the size bench.py runs them (config 1 in full: 4096 + 4096 states; configs 2-4
    at the largest state count that fits 7 state arrays), in the launch configuration bench.py
    times (default chunk, stream overlap on).  The oracle cannot step thousands of states, so: (i) the densities of
    ALL states against the oracle's densities_of, streamed in blocks (densities are sums over states); (ii) the
    potentials against the oracle's potentials_from those densities; (iii) H psi on a seeded sample of 64 states per
    species against the oracle's apply_h_with; (iv) after 3 starter + 2 ABM steps the invariants that hold at any
    size: norm and orthonormality defects, particle numbers and energy drift at the level SURVEY 8(c) states for
    incomplete sets."""
    from paper_2009_00745_b200 import lise
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    cfg = dict(inputs.CONFIGS[idx])
    shape = tuple(cfg["shape"])
    S = 64 * int(np.prod(shape))
    nwf = lise.capacity_states(shape, free, tuple(cfg["nwf"]))
    if sum(nwf) == 0 or free < 7 * S * sum(nwf) + 6 * 2 ** 30 or (idx == 1 and nwf != tuple(cfg["nwf"])):
        pytest.skip("not enough free device memory for the full-size workload")
    seed = inputs.SEED0 + idx
    # inputs first (the generator's workspace and the context's 7 arrays do not fit side by side at capacity)
    host = [inputs.make_block(cfg, q, nwf[q], 0, nwf[q], seed, "cuda").cpu() for q in (0, 1)]
    torch.cuda.empty_cache()
    g = lise.Lise(*shape, cfg["dx"], cfg["dt"], *nwf)
    oc = ref.RefContext(*shape, cfg["dx"], cfg["dt"], 1, 1)          # used for its stateless entry points only
    rng = np.random.default_rng(2009)
    dens_ref, sample = [], []
    for q in (0, 1):
        g.upload_wavefunctions(q, host[q])
        acc = np.zeros((14,) + shape)
        for f in range(0, nwf[q], 512):
            acc += oc.densities_of(host[q][f:f + 512].numpy()).reshape(acc.shape)
        dens_ref.append(acc)
        idxs = np.sort(rng.choice(nwf[q], size=64, replace=False))
        sample.append(host[q][torch.as_tensor(idxs)].contiguous().cuda())
    del host
    # tau, div J, curl j are grid derivatives of the accumulated fields: linear, so the block sum is exact
    for q in (0, 1):
        d_gpu = g.densities(q).cpu().numpy()
        assert field_rel(d_gpu, dens_ref[q]) < TOL_DENS, ("densities", q)
    pots = oc.potentials_from(dens_ref[0], dens_ref[1])
    for q in (0, 1):
        p_gpu = g.potentials(q).cpu().numpy()
        assert field_rel(p_gpu, np.asarray(pots[q]).reshape(p_gpu.shape)) < 1e-10, ("potentials", q)
        h_ref = oc.apply_h_with(np.asarray(pots[q]), sample[q].cpu().numpy()).reshape(sample[q].shape)
        h_gpu = g.apply_h(q, sample[q]).cpu().numpy()
        assert rel(h_gpu, h_ref) < 1e-12, ("H psi", q)
    o0 = g.observables()
    g.step(5)
    o1 = g.observables()
    assert o1["norm_defect"] < 1e-10 and o1["ortho_defect"] < 1e-10
    assert abs(o1["energy"] - o0["energy"]) < 1e-4 * abs(o0["energy"])
    for k in ("n_neutron", "n_proton"):
        assert abs(o1[k] - o0[k]) < 1e-4 * o0[k]
    g.close(); oc.close()


def test_reduce_hook_two_contexts_on_one_device():
    """state sharding through the product's own reduce hook (lise_set_reduce_hook), without a second GPU: two
    contexts on this device hold the two halves of the states of both species; their hooks meet at each density
    barrier and sum the two accumulator buffers in place, each on its own context's stream (event-ordered).  The
    sharded run must agree with the oracle on the full set and with a single-context run."""
    import threading
    from paper_2009_00745_b200 import lise, sharding
    cfg = dict(inputs.CONFIGS[1]); cfg["shape"] = (16, 16, 16)
    nwf = (26, 14)
    steps = 6                                        # 3 starter + 3 ABM
    psi = [inputs.make_species(cfg, q, nwf[q], seed=23) for q in (0, 1)]
    oc = ref.RefContext(*cfg["shape"], cfg["dx"], cfg["dt"], *nwf)
    for q in (0, 1):
        oc.set_wavefunctions(q, psi[q].numpy())
    oc.step(steps)
    single = lise.Lise(*cfg["shape"], cfg["dx"], cfg["dt"], *nwf)
    single.set_chunk(5)
    for q in (0, 1):
        single.set_wavefunctions(q, psi[q].cuda())
    single.step(steps)

    world = 2
    ranges = [[sharding.shard_range(nwf[q], world, r) for q in (0, 1)] for r in range(world)]
    streams = [torch.cuda.Stream() for _ in range(world)]
    ctxs = [lise.Lise(*cfg["shape"], cfg["dx"], cfg["dt"], ranges[r][0][1] - ranges[r][0][0],
                      ranges[r][1][1] - ranges[r][1][0], stream=streams[r]) for r in range(world)]
    meet = threading.Barrier(world)
    box = {"acc": [None] * world, "tmp": [None] * world,
           "ev1": [torch.cuda.Event() for _ in range(world)], "ev2": [torch.cuda.Event() for _ in range(world)]}
    calls = [0] * world

    def make_hook(r):
        def hook(t):                                  # runs under the context's stream (lise.py)
            o = 1 - r
            st = torch.cuda.current_stream()
            assert st.cuda_stream == streams[r].cuda_stream
            box["acc"][r] = t
            box["ev1"][r].record(st)
            meet.wait()                               # both partial accumulators are enqueued
            st.wait_event(box["ev1"][o])
            box["tmp"][r] = t + box["acc"][o]
            box["ev2"][r].record(st)
            meet.wait()                               # both sums are enqueued: the buffers may be overwritten
            st.wait_event(box["ev2"][o])
            t.copy_(box["tmp"][r])
            calls[r] += 1
        return hook

    errs, res = [], [None] * world

    def run(r):
        try:
            with torch.cuda.stream(streams[r]):
                c = ctxs[r]
                c.set_chunk(4); c.set_overlap(True)
                c.set_reduce_hook(make_hook(r))
                for q in (0, 1):
                    a, b = ranges[r][q]
                    c.set_wavefunctions(q, psi[q][a:b].cuda())
                c.step(steps)
                # every call that needs the potentials of y_n passes the density barrier (and the hook) once more:
                # both ranks make the same calls in the same order
                res[r] = dict(wf=[c.get_wavefunctions(q).cpu().numpy() for q in (0, 1)],
                              dens=[c.densities(q).cpu().numpy() for q in (0, 1)], energy=c.observables()["energy"])
                streams[r].synchronize()
        except Exception as exc:                      # pragma: no cover
            errs.append(exc)
            meet.abort()

    th = [threading.Thread(target=run, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errs, errs
    assert calls[0] == calls[1] and calls[0] >= 2 * steps
    for q in (0, 1):
        w_ref = oc.get_wavefunctions(q)
        w_one = single.get_wavefunctions(q).cpu().numpy()
        w_sh = np.concatenate([res[r]["wf"][q] for r in range(world)])
        assert rel(w_sh, w_ref) < TOL_WF, ("sharded vs oracle", q)
        assert rel(w_sh, w_one) < 1e-12, ("sharded vs single context", q)
        d_ref = oc.densities(q)
        for r in range(world):                        # replicated grid fields: every rank holds the global densities
            assert field_rel(res[r]["dens"][q], d_ref) < TOL_DENS, ("densities", q, r)
    e_ref = oc.observables()["energy"]
    for r in range(world):
        assert abs(res[r]["energy"] - e_ref) < TOL_E * abs(e_ref)
    for c in ctxs:
        c.close()
    single.close(); oc.close()


def test_stream_overlap_does_not_change_results():
    """lise_set_overlap (update kernels on a second stream beside the tensor-core kernels, several chunks in flight,
    densities per group of chunks) is a scheduling choice: bit-identical wavefunctions, densities and energy."""
    from paper_2009_00745_b200 import lise
    cfg = dict(inputs.CONFIGS[1]); cfg["shape"] = (16, 16, 16)
    nwf = (29, 23)
    psi = [inputs.make_species(cfg, q, nwf[q], seed=11).cuda() for q in (0, 1)]
    res = []
    for overlap in (True, False):
        g = lise.Lise(*cfg["shape"], cfg["dx"], cfg["dt"], *nwf)
        g.set_chunk(4)                               # many chunks, ragged tail
        g.set_overlap(overlap)
        for q in (0, 1):
            g.set_wavefunctions(q, psi[q])
        g.step(6)
        res.append(([g.get_wavefunctions(q).cpu().numpy() for q in (0, 1)],
                    [g.densities(q).cpu().numpy() for q in (0, 1)], g.observables()["energy"]))
        g.close()
    for q in (0, 1):
        assert np.array_equal(res[0][0][q], res[1][0][q])
        assert np.array_equal(res[0][1][q], res[1][1][q])
    assert res[0][2] == res[1][2]


def test_edge_cases_and_errors():
    from paper_2009_00745_b200 import lise
    import ctypes as C
    lib = lise.load()
    h = C.c_void_p()
    assert lib.lise_create(12, 12, 11, 1.0, 0.05, 4, 0, C.byref(h)) == -1          # odd lattice size
    assert lib.lise_create(12, 12, 12, -1.0, 0.05, 4, 0, C.byref(h)) == -1         # bad spacing
    assert lib.lise_create(12, 12, 12, 1.0, 0.05, 4, 0, None) == -1
    g = lise.Lise(12, 12, 12, 1.5, 0.05, 4, 3)
    with pytest.raises(lise.LiseError):
        g.step(1)                                                                    # wavefunctions not set
    with pytest.raises(lise.LiseError):
        g.densities(0)
    g.close()
    # empty proton species and zero steps are fine
    cfg = dict(inputs.CONFIGS[0])
    psi = inputs.make_species(cfg, 0, 3, seed=1).cuda()
    g = lise.Lise(*cfg["shape"], cfg["dx"], 0.05, 3, 0)
    g.set_wavefunctions(0, psi)
    g.step(0)
    assert torch.equal(g.get_wavefunctions(0), psi)
    assert float(g.densities(1).abs().max()) == 0.0
    g.close()


@pytest.mark.parametrize("nwf", [(1, 0), (0, 2), (1, 1)])
def test_degenerate_state_counts(nwf):
    """fewer states than state groups (most plane-owner CTAs, and one of the two unit pipelines of the xz kernel, have no
    work), a single state, protons only (Coulomb on, no neutron at all): 3 starter + 3 ABM steps against the oracle."""
    from paper_2009_00745_b200 import lise
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (12, 12, 12)
    psi = [inputs.make_species(cfg, q, nwf[q], seed=77 + q) for q in (0, 1)]
    po = ref.default_params(); pg = lise.default_params()
    po.coulomb = pg.coulomb = 1 if nwf[1] else 0
    oc = ref.RefContext(*cfg["shape"], cfg["dx"], 0.05, *nwf, params=po)
    gc = lise.Lise(*cfg["shape"], cfg["dx"], 0.05, *nwf, params=pg)
    for q in (0, 1):
        oc.set_wavefunctions(q, psi[q].numpy())
        gc.set_wavefunctions(q, psi[q].cuda())
    oc.step(6); gc.step(6)
    for q in (0, 1):
        if nwf[q] == 0:
            assert float(gc.densities(q).abs().max()) == 0.0
            continue
        assert rel(gc.get_wavefunctions(q).cpu().numpy(), oc.get_wavefunctions(q)) < TOL_WF
        assert field_rel(gc.densities(q).cpu().numpy(), oc.densities(q)) < TOL_DENS
    eo, eg = oc.observables(), gc.observables()
    assert abs(eg["energy"] - eo["energy"]) < TOL_E * abs(eo["energy"])
    # H applied to zero states is a no-op
    q = 0 if nwf[0] else 1
    empty = torch.zeros((0, 4) + tuple(cfg["shape"]), dtype=torch.complex128, device="cuda")
    assert gc.apply_h(q, empty).shape[0] == 0
    gc.close(); oc.close()


def test_defects_of_a_non_orthonormal_set():
    """norm and orthonormality defects of lise_observables on a set with a planted overlap sin(0.3) and a planted
    norm 1.05^2: the closed-form values (the oracle is pinned to the same ones on the CPU)."""
    import math
    from paper_2009_00745_b200 import lise
    from tests.test_oracle_pins import _defective_set
    shape, dx, nwf, theta, scale = (8, 8, 8), 1.5, 6, 0.3, 1.05
    psi = _defective_set(shape, dx, nwf, theta, scale)
    g = lise.Lise(*shape, dx, 0.05, nwf, 0)
    g.set_wavefunctions(0, torch.from_numpy(psi).cuda())
    g.set_wavefunctions(1, torch.zeros((0, 4) + shape, dtype=torch.complex128, device="cuda"))
    o = g.observables()
    assert abs(o["norm_defect"] - (scale ** 2 - 1.0)) < 1e-12
    assert abs(o["ortho_defect"] - math.sin(theta)) < 1e-12
    g.close()


def _white_noise_states(shape, dx, nwf, seed):
    """every component of every state drawn from uniform(-1, 1) + i uniform(-1, 1) at every lattice point
    (then normalised to dV sum |psi|^2 = 1): all wavevectors up to and including the Nyquist planes carry full weight."""
    rng = np.random.default_rng(seed)
    psi = rng.uniform(-1.0, 1.0, (nwf, 4) + tuple(shape)) + 1j * rng.uniform(-1.0, 1.0, (nwf, 4) + tuple(shape))
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2, 3, 4), keepdims=True) * dx ** 3)
    return np.ascontiguousarray(psi)


# one lattice per kernel family: whole-state FFT units (24^3), 2-spinor FFT units with the pairing block in the xz
# kernel (32^3), block-diagonalised circulant on the fp64 tensor cores (24^2 x 48), generic DFMA kernels (6 x 10 x 12)
@pytest.mark.parametrize("shape,line_op", [((24, 24, 24), "fft"), ((32, 32, 32), "fft"), ((24, 24, 48), "dmma"), ((6, 10, 12), "dense")])
def test_white_noise_states_reach_the_nyquist_branch_of_every_kernel_family(shape, line_op):
    """The band-limited generator of the other cases feeds the Nyquist planes (D zeroed, D2 kept) only
    through the envelope's leakage; white noise (the paper's own noise distribution, L685) puts full weight there.
    lise_densities, lise_potentials and lise_apply_h of such states against the oracle, in every kernel family."""
    from paper_2009_00745_b200 import lise
    dx, nwf = 1.25, (6, 4)
    psi = [_white_noise_states(shape, dx, nwf[q], 685 + q) for q in (0, 1)]
    oc = ref.RefContext(*shape, dx, 0.05, *nwf)
    gc = lise.Lise(*shape, dx, 0.05, *nwf)
    assert gc.line_operator() == line_op
    for q in (0, 1):
        oc.set_wavefunctions(q, psi[q]); gc.set_wavefunctions(q, torch.from_numpy(psi[q]).cuda())
    for q in (0, 1):
        assert field_rel(gc.densities(q).cpu().numpy(), oc.densities(q)) < TOL_DENS, (shape, "densities", q)
        assert field_rel(gc.potentials(q).cpu().numpy(), oc.potentials(q)) < 1e-10, (shape, "potentials", q)
        h_ref = oc.apply_h(q, psi[q])
        h_gpu = gc.apply_h(q, torch.from_numpy(psi[q]).cuda()).cpu().numpy()
        assert rel(h_gpu, h_ref.reshape(h_gpu.shape)) < 1e-12, (shape, "H psi", q)
    gc.close(); oc.close()


def test_line_operator_families_agree_and_can_be_chosen_at_creation():
    """lise_create_with_line_operator: the generic DFMA kernels against the FFT kernels on 24^3 (densities, potentials,
    H psi, 3 starter + 1 ABM steps) and against the tensor-core kernels on 24^2 x 48 (H psi); families that were not
    instantiated for a lattice, and unknown names, are refused with a message."""
    from paper_2009_00745_b200 import lise
    cfg = dict(inputs.CONFIGS[1])
    nwf = (12, 8)
    psi = [inputs.make_species(cfg, q, nwf[q], seed=77).cuda() for q in (0, 1)]
    ctx = {}
    for name in ("fft", "dense"):
        g = lise.Lise(*cfg["shape"], cfg["dx"], cfg["dt"], *nwf, line_operator=name)
        assert g.line_operator() == name
        for q in (0, 1):
            g.set_wavefunctions(q, psi[q])
        ctx[name] = g
    a, b = ctx["fft"], ctx["dense"]
    for q in (0, 1):
        assert field_rel(a.densities(q).cpu().numpy(), b.densities(q).cpu().numpy()) < TOL_DENS
        assert field_rel(a.potentials(q).cpu().numpy(), b.potentials(q).cpu().numpy()) < 1e-10
        assert rel(a.apply_h(q, psi[q]).cpu().numpy(), b.apply_h(q, psi[q]).cpu().numpy()) < 1e-12
    a.step(4); b.step(4)
    for q in (0, 1):
        assert rel(a.get_wavefunctions(q).cpu().numpy(), b.get_wavefunctions(q).cpu().numpy()) < TOL_WF
    ea, eb = a.observables()["energy"], b.observables()["energy"]
    assert abs(ea - eb) < TOL_E * abs(eb)
    a.close(); b.close()
    shape = (24, 24, 48)
    cfg3 = dict(inputs.CONFIGS[3]); cfg3["shape"] = shape
    psi3 = [inputs.make_species(cfg3, q, 5, seed=78).cuda() for q in (0, 1)]
    out = {}
    for name in ("dmma", "dense"):
        g = lise.Lise(*shape, cfg3["dx"], cfg3["dt"], 5, 5, line_operator=name)
        assert g.line_operator() == name
        for q in (0, 1):
            g.set_wavefunctions(q, psi3[q])
        out[name] = [g.apply_h(q, psi3[q]).cpu().numpy() for q in (0, 1)]
        g.close()
    for q in (0, 1):
        assert rel(out["dmma"][q], out["dense"][q]) < 1e-12
    with pytest.raises(lise.LiseError, match="no dmma kernels"):
        lise.Lise(24, 24, 24, 1.25, 0.05, 2, 2, line_operator="dmma")
    with pytest.raises(lise.LiseError, match="no fft kernels"):
        lise.Lise(6, 10, 12, 1.25, 0.05, 2, 2, line_operator="fft")
    with pytest.raises(lise.LiseError, match="unknown line operator"):
        lise.Lise(24, 24, 24, 1.25, 0.05, 2, 2, line_operator="cufft")
    g = lise.Lise(24, 24, 24, 1.25, 0.05, 2, 2, line_operator="auto")
    assert g.line_operator() == "fft"
    g.close()


@pytest.mark.parametrize("shape", [(24, 24, 24), (32, 32, 32), (24, 24, 48), (6, 10, 12)])
def test_caller_buffers_are_not_overrun(shape):
    """compute-sanitizer is closed on this GPU pool (profiles/r3_sanitizer.md), so the bounds of the caller-owned buffers
    are checked here instead: every output of the C ABI is a window inside a larger allocation filled with a canary, the
    inputs sit between canaries too, and after lise_densities / lise_potentials / lise_apply_h / lise_step /
    lise_get_wavefunctions on a ragged state count the canaries on both sides must be untouched -- for each kernel
    family (FFT whole-state, FFT 2-spinor, tensor-core, generic)."""
    from paper_2009_00745_b200 import lise
    cfg = dict(inputs.CONFIGS[1]); cfg["shape"] = shape
    nwf, nxyz, pad = (7, 5), int(np.prod(shape)), 4096
    CAN = complex(-7.25e300, 3.5e299)

    def window(count, dtype):
        big = torch.full((count + 2 * pad,), CAN if dtype == torch.complex128 else CAN.real, dtype=dtype, device="cuda")
        return big, big[pad:pad + count]

    def intact(big, count):
        edge = torch.cat([big[:pad], big[pad + count:]])
        want = CAN if big.dtype == torch.complex128 else CAN.real
        return bool((edge == want).all())

    g = lise.Lise(*shape, cfg["dx"], cfg["dt"], *nwf)
    g.set_chunk(3)                                                  # ragged: 3 + 3 + 1 and 3 + 2 states
    for q in (0, 1):
        n = nwf[q] * 4 * nxyz
        big_in, w_in = window(n, torch.complex128)
        w_in.copy_(inputs.make_species(cfg, q, nwf[q], seed=90).reshape(-1).cuda())
        g.set_wavefunctions(q, w_in.reshape((nwf[q], 4) + shape))
        assert intact(big_in, n)
    g.step(4)                                                       # 3 starter + 1 ABM step on the internal buffers
    for q in (0, 1):
        n = nwf[q] * 4 * nxyz
        for call in (g.densities, g.potentials):
            big, w = window(14 * nxyz, torch.float64)
            call(q, out=w.reshape((14,) + shape))
            torch.cuda.synchronize()
            assert intact(big, 14 * nxyz) and bool(torch.isfinite(w).all()), (call.__name__, q)
        big_o, w_o = window(n, torch.complex128)
        g.get_wavefunctions(q, out=w_o.reshape((nwf[q], 4) + shape))
        big_h, w_h = window(n, torch.complex128)
        g.apply_h(q, w_o, out=w_h)
        torch.cuda.synchronize()
        assert intact(big_o, n) and intact(big_h, n), q
        assert bool(torch.isfinite(w_h.real).all()) and float(w_h.abs().max()) < 1e6
    o = g.observables()
    assert o["norm_defect"] < 1e-10 and np.isfinite(o["energy"])
    g.close()
