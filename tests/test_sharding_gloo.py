"""Multi-process (world_size 2, gloo, CPU) test of the state-sharding host logic:
shard ranges partition the states, the density all-reduce sums the ranks' partial accumulators, and the
per-rank defect maxima combine.  The partial accumulators here come from the oracle's densities of each
rank's own states (densities are sums over states, Eq. 3), so the test also checks the property
the sharded GPU path relies on: sum over ranks of shard densities == densities of the full set."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2009_00745_b200 import inputs, sharding


def test_shard_ranges_partition():
    for nwf in (0, 1, 7, 128, 4097):
        for world in (1, 2, 3, 8):
            edges = [sharding.shard_range(nwf, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == nwf
            for a, b in zip(edges, edges[1:]):
                assert a[1] == b[0]
            counts = sharding.shard_counts(nwf, world)
            assert sum(counts) == nwf and max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        sharding.shard_range(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, nwf, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import ref
        cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (8, 6, 8)
        psi = inputs.make_species(cfg, 0, nwf, seed=11)
        first, last = sharding.shard_range(nwf, world, rank)
        oc = ref.RefContext(*cfg["shape"], cfg["dx"], cfg["dt"], last - first, 0)
        oc.set_wavefunctions(0, psi[first:last].numpy())
        # rows of Table 2 that are linear in the accumulators: n, s, j, kappa (tau, div J, curl j are
        # grid derivatives of sums, linear as well)
        part = torch.from_numpy(np.ascontiguousarray(oc.densities(0))).clone()
        oc.close()
        sharding.allreduce_sum_(part)
        obs = sharding.global_observables({"norm_defect": 1e-3 * (rank + 1), "ortho_defect": 1e-4 * (world - rank), "energy": 1.0})
        if rank == 0:
            np.save(os.path.join(out_dir, "summed.npy"), part.numpy())
            np.save(os.path.join(out_dir, "obs.npy"), np.array([obs["norm_defect"], obs["ortho_defect"]]))
    finally:
        dist.destroy_process_group()


def test_density_allreduce_world2(tmp_path):
    from oracle import ref
    ref.build()
    world, nwf = 2, 7
    mp.spawn(_worker, args=(world, _free_port(), nwf, str(tmp_path)), nprocs=world, join=True)
    summed = np.load(tmp_path / "summed.npy")
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (8, 6, 8)
    psi = inputs.make_species(cfg, 0, nwf, seed=11)
    oc = ref.RefContext(*cfg["shape"], cfg["dx"], cfg["dt"], nwf, 0)
    oc.set_wavefunctions(0, psi.numpy())
    full = oc.densities(0)
    oc.close()
    assert np.abs(summed - full).max() <= 1e-12 * np.abs(full).max()
    obs = np.load(tmp_path / "obs.npy")
    assert obs[0] == pytest.approx(2e-3) and obs[1] == pytest.approx(2e-4)


class _FakeCtx:
    """stands in for lise.Lise in attach(): the fields and setters attach touches, no GPU."""

    class _P:
        def __init__(self, coulomb):
            self.coulomb = coulomb

    def __init__(self, nwf, requested):
        self.nwf = nwf
        self.coulomb_requested = requested
        self.params = self._P(requested if nwf[1] > 0 else 0)       # Lise.__init__: no proton states -> Coulomb off
        self.hook = None

    def set_params(self, p):
        self.params = p
        self.coulomb_requested = int(p.coulomb)

    def set_reduce_hook(self, fn):
        self.hook = fn


def _attach_worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        res = []
        nwf = (4, 3) if rank == 0 else (4, 0)                       # rank 1 owns no proton state
        for requested, override, global_nwf in ((1, None, None), (0, None, None), (1, None, (8, 3)), (0, True, None), (1, False, None)):
            c = _FakeCtx(nwf, requested)
            sharding.attach(c, global_nwf=global_nwf, coulomb=override)
            res.append(c.params.coulomb)
            assert c.hook is not None
        c = _FakeCtx((4, 0), 1)                                     # no rank holds protons: off everywhere
        sharding.attach(c)
        res.append(c.params.coulomb)
        c = _FakeCtx(nwf, 1 if rank == 0 else 0)                    # ranks disagree: refused on every rank
        try:
            sharding.attach(c)
            res.append(-1)
        except ValueError:
            res.append(9)
        np.save(os.path.join(out_dir, f"attach{rank}.npy"), np.array(res))
    finally:
        dist.destroy_process_group()


def test_attach_decides_coulomb_from_the_request_and_the_global_proton_count(tmp_path):
    """a context configured with coulomb = 0 must stay off; a rank without proton states follows the others."""
    mp.spawn(_attach_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    want = [1, 0, 1, 1, 0, 0, 9]
    for rank in (0, 1):
        assert list(np.load(tmp_path / f"attach{rank}.npy")) == want, rank
    # single process, no process group: the local counts decide
    c = _FakeCtx((4, 0), 1); sharding.attach(c); assert c.params.coulomb == 0
    c = _FakeCtx((4, 2), 0); sharding.attach(c); assert c.params.coulomb == 0 and c.coulomb_requested == 0
    c = _FakeCtx((4, 2), 1); sharding.attach(c); assert c.params.coulomb == 1
