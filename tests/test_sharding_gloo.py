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
