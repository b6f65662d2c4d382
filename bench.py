#!/usr/bin/env python
"""Benchmark of the TDSLDA time step (BASELINE.json metric: qp-wavefunction updates/sec, fp64).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config I]

A "step" is one Adams-Bashforth-Milne predictor-modifier-corrector step (two H evaluations, two density
barriers, Eq. 78) of EVERY quasiparticle state of both species of the workload; the starter
(3 series-expansion steps) and lise_observables are outside the timed region.  value = states x K / time.
N > 1 (torchrun, one rank per GPU): weak scaling, every rank owns the full per-GPU state count, one
NCCL all-reduce of the density accumulators per barrier.  `--impl reference` times the CPU oracle
(oracle/, as it stands) on a bounded sample of the same workload on the host cores.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "qp-wavefunction updates/sec (fp64 TDSLDA steps)"
UNIT = "qpwf-updates/s"


def read_peaks():
    """measured denominators written by the driver, else the fallback of B200_PROFILING.md."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def measured_traffic(cls, workload, states_per_launch):
    """DRAM bytes per launch of kernel class `cls` from the committed ncu capture (profiles/r2_traffic.md: bytes per
    state on the config-1 lattice, `ncu --set full`, dram__bytes_read.sum + dram__bytes_write.sum), or None for other
    workloads / when the file is absent.  Not measured in this run: a number taken under ncu is never a bench value."""
    if not workload.startswith("config1"):
        return None
    path = os.path.join(ROOT, "profiles", "r2_traffic.md")
    try:
        for line in open(path):
            cells = [c.strip() for c in line.strip().strip("|").split("|")]
            if len(cells) == 5 and cells[0] == cls:
                return float(cells[4]) * states_per_launch
    except OSError:
        pass
    return None


class ClockSampler:
    """nvidia-smi polled every 50 ms in the background; started BEFORE the warm-up steps (its start-up takes a few
    hundred ms) and filtered to the timed region by its own timestamps."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self, t0, t1):
        """samples with t0 <= timestamp <= t1 (wall clock of the timed region); if the region was shorter than the polling
        interval, the samples since the sampler started (warm-up steps: the same load) are used and `window` says so."""
        import datetime
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        rows = []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(parts[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                rows.append((ts, float(parts[1]), float(parts[2]), float(parts[3]),
                             [n for n, v in zip(names, parts[4:8]) if v.lower().startswith("active")]))
            except ValueError:
                continue
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        inside = [r for r in rows if t0 - 0.025 <= r[0] <= t1 + 0.025]
        window = "timed region"
        if not inside:
            inside = [r for r in rows if r[0] <= t1 + 0.025]
            window = "warm-up + timed region (timed region shorter than the polling interval)"
        if inside:
            sm = sorted(r[1] for r in inside)
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(r[2] for r in inside),
                       reasons=sorted({n for r in inside for n in r[4]}), samples=len(inside),
                       power_w_max=max(r[3] for r in inside), window=window)
        return out


def workload(idx, nwf_override=None):
    from paper_2009_00745_b200 import inputs
    cfg = dict(inputs.CONFIGS[idx])
    nwf = tuple(nwf_override) if nwf_override else tuple(cfg["nwf"])
    return cfg, nwf


# ---- ALGORITHMIC work per kernel class, per state and evaluation (two evaluations per ABM step) ----
# flops: an axis pass = one 1-D transform of every line of one component along one axis = 5 N log2 N per line of N
# points, i.e. 5 log2 N per lattice point.  H-apply: 4 components x 6 passes per axis (inner 1 forward + 2 inverse,
# outer 2 forward + 1 inverse); densities: 2 v-components x 3 passes per axis; pointwise: 545 (H-apply incl. the k-space
# multipliers and pairing, two thirds on the yz kernel), 120 (density accumulators, same split), 16 (eta), 270 per STEP
# for the ABM linear combinations.  Sum over a step = 300 (log2 Nx + log2 Ny + log2 Nz) + 1600 per point, the survey's figure.
# bytes: 15 S per step (S = 64 Nxyz): X read once per evaluation (charged to the yz kernel), phase 1: 5 history reads
# + 4 writes, phase 2: 2 reads + 2 writes (charged to the update).  W = H psi is NOT counted: it should stay on chip.
def algorithmic_model(shape):
    lx, ly, lz = (math.log2(n) for n in shape)
    return {
        "happly_yz": dict(flop=4 * 6 * 5.0 * (ly + lz) + 545.0 * 2 / 3, S=1.0),
        "happly_xz": dict(flop=4 * 6 * 5.0 * lx + 545.0 / 3 + 16.0, S=0.0),
        "update": dict(flop=135.0, S=6.5),                          # mean of 9 S (evaluation 1) and 4 S (evaluation 2)
        "dens_yz": dict(flop=2 * 3 * 5.0 * (ly + lz) + 120.0 * 2 / 3, S=0.0),
        "dens_x": dict(flop=2 * 3 * 5.0 * lx + 120.0 / 3, S=0.0),
        "grid": dict(flop=0.0, S=0.0),
    }


def step_flops_per_point(shape):
    return 300.0 * sum(math.log2(n) for n in shape) + 1600.0


# ---- EXECUTED fp64-pipe work of this build (a model of what the kernels run, not the roofline numerator) ----
# FFT line operator: the generated codelets' instruction counts (lise_line_operator_cost: inner + outer per real line
# of N points = 4 operator applications on one real part); DMMA line operator: 256 FMA slots per m8n8k4 tile,
# dmma_tiles(N) tiles per 8 real columns and operator application; + pointwise slots.  1 slot = 1 fp64 instruction lane.
def dmma_tiles(n):
    if n % 8 == 0 and 16 <= n <= 64:
        r = n // 8
        nreal = 1 + (1 if r % 2 == 0 else 0)
        return 2 * nreal + 8 * ((r - 1) // 2)
    return ((n + 7) // 8) * (n // 4)                               # plain circulant


def executed_model(shape, line_op, lise):
    nx, ny, nz = shape

    def dmma_axis(n):                                              # slots per complex point, component and axis (4 applications)
        return 4 * dmma_tiles(n) * 256.0 / (4.0 * n)

    def fft_axis(n):
        c = lise.line_operator_cost(n)
        return 2.0 * (c[0] + c[1]) / n if c[0] else dmma_axis(n)
    pw = 50.0                                                      # pointwise + small transforms per point, component and axis
    fft_yz = line_op == "fft"
    fft_xz = fft_yz                                                # lise.cu make_v6_set: both H-apply kernels of an "fft" set run FFT lines
    ay = (fft_axis if fft_yz else dmma_axis)
    ax = (fft_axis if fft_xz else dmma_axis)
    return {
        "happly_yz": 4 * (ay(ny) + ay(nz) + 2 * pw) + 4 * 12,
        "happly_xz": 4 * (ax(nx) + pw),
        "update": 40.0,
        "dens_yz": 2 * (0.5 * (dmma_axis(ny) + dmma_axis(nz)) + 20) + 20,
        "dens_x": 2 * (0.5 * dmma_axis(nx) + 10),
        "grid": 0.0,
    }


def run_workload(args, cfg_idx, nwf_req, env, primary):
    """one workload on this rank's GPU: setup, starter, warm-up, K timed ABM steps, per-class times; returns a dict
    (rank 0) or None."""
    import torch
    import torch.distributed as dist
    from paper_2009_00745_b200 import inputs, lise, sharding
    world, rank, dev, local = env["world"], env["rank"], env["dev"], env["local"]
    cfg, nwf = workload(cfg_idx, nwf_req)
    shape = tuple(cfg["shape"]); nxyz = shape[0] * shape[1] * shape[2]
    S = 64.0 * nxyz
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info(dev)
    req = nwf
    nwf = lise.capacity_states(shape, free, nwf)                 # 7 state arrays must fit
    if sum(nwf) == 0:                                             # (0, 0): not even 256 states per requested species fit
        why = f"does not fit: {free / 2 ** 30:.1f} GiB free for {req[0]} + {req[1]} states of {S / 2 ** 20:.2f} MB x 7 arrays"
        if primary:
            raise SystemExit(f"bench.py: config {cfg_idx} {why}")
        return {"skipped": why, "config": {"workload": f"config{cfg_idx}", "shape": list(shape), "nwf_requested": list(req)}} if rank == 0 else None
    tot = (nwf[0] * world, nwf[1] * world)                        # weak scaling: global counts
    seed = inputs.SEED0 + cfg_idx
    steps = args.steps                                            # every workload of the line gets the full --steps

    # inputs first, parked in pinned host memory: the generator's workspace and the context's 7 arrays do not fit side
    # by side at capacity; the host copies are also the end-to-end leg's mirror
    t0 = time.time()
    host = []
    for q in (0, 1):
        if nwf[q] == 0:
            host.append(None)
            continue
        psi = inputs.make_block(cfg, q, tot[q], rank * nwf[q], nwf[q], seed, dev)
        h = torch.empty(psi.shape, dtype=torch.complex128, pin_memory=True)
        h.copy_(psi)
        host.append(h)
        del psi
    torch.cuda.empty_cache()
    g = lise.Lise(*shape, cfg["dx"], cfg["dt"], nwf[0], nwf[1])
    if world > 1:
        sharding.attach(g, global_nwf=tot, coulomb=bool(cfg["coulomb"]))   # the workload's flag, the same on every rank
    if args.chunk:
        g.set_chunk(args.chunk)
    if args.dgroup:
        g.set_density_group(args.dgroup)
    for q in (0, 1):
        if host[q] is not None:
            g.upload_wavefunctions(q, host[q])
        else:
            g.set_wavefunctions(q, torch.zeros((0, 4) + shape, dtype=torch.complex128, device=dev))
    torch.cuda.synchronize()
    t_setup = time.time() - t0

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    nstates = nwf[0] + nwf[1]
    g.step(3)                                   # series-expansion starter: outside the timed region
    sampler = ClockSampler(local) if rank == 0 else None
    for _ in range(args.warmup):
        g.step(1)
    barrier()
    l0 = g.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    wall0 = time.time()
    ev0.record()
    g.step(steps)
    ev1.record()
    barrier()
    wall1 = time.time()
    wall = wall1 - wall0
    ms = ev0.elapsed_time(ev1)
    launches = g.launch_count() - l0
    clocks = sampler.stop(wall0, wall1) if sampler else None
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t[0])
    value = nstates * world * steps / (ms * 1e-3)
    obs = g.observables()

    # ---- per-kernel-class device times (CUDA events inside the library, on the launching stream) ----
    # with the two-stream overlap off: a class time is then that kernel running alone, which is what a per-kernel
    # roofline needs (overlapped, the update and the H-apply kernels share SMs and stretch each other)
    psteps = max(1, min(steps, 2))
    g.set_overlap(False)
    g.profile(True)
    g.step(psteps)
    prof = g.profile_read()
    g.profile(False)
    g.set_overlap(True)

    # ---- end to end through the C-ABI with HOST buffers ----
    e2e = None
    if args.e2e and primary:
        for q in (0, 1):
            if host[q] is not None:
                g.download_wavefunctions(q, host[q])            # host mirror of y_n
        barrier()
        w0 = time.time()
        for _ in range(steps):
            for q in (0, 1):
                if host[q] is not None:
                    g.upload_wavefunctions(q, host[q], keep_history=True)   # H2D of the step's input
            g.step(1)
            for q in (0, 1):
                if host[q] is not None:
                    g.download_wavefunctions(q, host[q])        # D2H of the step's result (y_{n+1}); synchronises
        barrier()
        w = time.time() - w0
        if world > 1:
            t = torch.tensor([w], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            w = float(t[0])
        nbytes = sum(h.numel() * 16 for h in host if h is not None)
        e2e = {"value": nstates * world * steps / w, "unit": UNIT,
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes}
    del host
    line_op = g.line_operator()
    if rank != 0:
        g.close()
        return None

    # ---- rooflines: algorithmic flops and bytes over the measured peaks ----
    hbm_gbs, hbm_src = read_peaks()
    fp64_tf = env["fp64_tf"]
    alg = algorithmic_model(shape)
    exe = executed_model(shape, line_op, lise)
    tot_ms = sum(v[0] for v in prof.values())
    top = max((k for k in prof if k != "grid"), key=lambda k: prof[k][0])
    top_ms, top_n = prof[top]
    states_per_launch = nstates * psteps * 2.0 / max(top_n, 1)       # every state passes each class twice per step
    flop_per_launch = alg[top]["flop"] * nxyz * states_per_launch
    bytes_per_launch = alg[top]["S"] * S * states_per_launch
    avg_s = top_ms * 1e-3 / max(top_n, 1)
    t_hbm = bytes_per_launch / (hbm_gbs * 1e9)
    t_alu = flop_per_launch / (fp64_tf * 1e12)
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": flop_per_launch / avg_s * 1e-12, "peak": fp64_tf, "unit": "TFLOP/s",
                "peak_source": "measured here: DFMA microbenchmark (lise_measure_fp64_peak), 2 flop per fp64 pipe slot; "
                               "nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
                "numerator": "SURVEY 8(d) algorithmic flops (5 N log2 N per line transform + pointwise), not executed work"}
    else:
        roof = {"bound": "hbm", "achieved": bytes_per_launch / avg_s * 1e-9, "peak": hbm_gbs, "unit": "GB/s",
                "peak_source": hbm_src, "numerator": "SURVEY 8(d) algorithmic bytes"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["kernel"] = top
    roof["avg_launch_ms"] = avg_s * 1e3
    roof["share_of_step"] = top_ms / tot_ms if tot_ms > 0 else None
    roof["executed_tflops"] = exe[top] * 2.0 * nxyz * states_per_launch / avg_s * 1e-12
    roof["executed_note"] = "model of the fp64-pipe slots this build executes (codelet / DMMA tile counts), 2 flop per slot"
    roof["traffic"] = measured_traffic(top, cfg["name"], states_per_launch)
    roof["traffic_source"] = "profiles/r2_traffic.md (committed ncu --set full capture, bytes per state x states per launch)"
    roof["classes_ms_per_step"] = {k: v[0] / psteps for k, v in prof.items()}
    roof["classes_frac_of_fp64_peak"] = {k: (alg[k]["flop"] * nxyz * nstates * 2.0 / (v[0] / psteps * 1e-3) / (fp64_tf * 1e12)
                                             if v[0] > 0 else None) for k, v in prof.items()}
    roof["classes_note"] = "per-class device time with the update/H-apply stream overlap off; the timed region runs with it on"
    step_bytes = 15.0 * S                                              # B_min = 960 Nxyz per qpwf-update
    step_flop = step_flops_per_point(shape) * nxyz
    per_gpu = value / world
    hbm_frac = per_gpu * step_bytes / (hbm_gbs * 1e9)
    fp64_frac = per_gpu * step_flop / (fp64_tf * 1e12)
    step_roof = {"hbm_bytes_per_update": step_bytes, "flop_per_update": step_flop,
                 "hbm_frac_of_measured": hbm_frac, "hbm_frac_of_8TBs": per_gpu * step_bytes / 8e12,
                 "fp64_frac_of_measured": fp64_frac, "fp64_frac_of_nominal_37.2": per_gpu * step_flop / 37.2e12,
                 "headline_frac": min(hbm_frac, fp64_frac),
                 "headline_note": "SURVEY 8(d): min(HBM fraction, fp64 fraction) of the whole step, both of measured peaks",
                 "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": hbm_src, "fp64_peak_tflops_measured": fp64_tf}
    par = "single GPU"
    if world > 1:
        par = (f"state-sharded x{world}, weak scaling: every rank owns {nstates} states, each shard orthonormalised on its "
               "own (the union is not one orthonormal set; densities are additive either way)")
    out = {"value": value, "ms_per_step": ms / steps, "steps": steps,
           "config": {"workload": cfg["name"], "lattice": list(shape), "dx_fm": cfg["dx"], "dt_fm_c": cfg["dt"],
                      "states_per_gpu": list(nwf), "states_requested": list(req), "coulomb": bool(cfg["coulomb"] and tot[1] > 0),
                      "parallelism": par,
                      "l2": "inputs larger than L2 (7 state arrays = %.1f GB resident)" % (7 * S * nstates / 1e9),
                      "line_operator": line_op, "setup_s": round(t_setup, 1)},
           "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "step_roofline": step_roof,
           "wall_s_timed_region": wall,
           "observables": {k: obs[k] for k in ("energy", "n_neutron", "n_proton", "norm_defect", "ortho_defect", "step")}}
    g.close()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2009_00745_b200 import lise

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` without a launcher: re-run this command line under torch.distributed.run, one rank
        # per GPU, so that a scaling run can never silently measure one GPU and label it N
        import socket
        with socket.socket() as so:
            so.bind(("127.0.0.1", 0))
            port = so.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.stdout.flush()
        os.execv(sys.executable, cmd)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus != world:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={world} ranks")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    env = dict(world=world, rank=rank, local=local, dev=dev, fp64_tf=lise.measure_fp64_peak(1.5) if rank == 0 else 0.0)
    res = run_workload(args, args.config, args.nwf, env, primary=True)
    also = []
    if args.also and args.nwf is None:
        for idx in args.also:
            if idx != args.config:
                r = run_workload(args, idx, None, env, primary=False)
                if r is not None:
                    also.append(r)
    if rank == 0:
        out = {"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
               "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "f64", "data": "synthetic"}
        for k in ("config", "clocks", "e2e", "gpu_launches", "roofline", "step_roofline", "wall_s_timed_region", "observables"):
            out[k] = res[k]
        # the other workload the target names (32^3), same invocation: its own clocks, rooflines, state counts
        out["also"] = [r if "skipped" in r else
                       {"metric": METRIC, "unit": UNIT, **{k: r[k] for k in ("value", "ms_per_step", "steps", "config", "clocks",
                        "gpu_launches", "roofline", "step_roofline", "observables")}} for r in also]
        if args.cpu_baseline and world == 1:
            from paper_2009_00745_b200 import inputs
            out["cpu_baseline"] = cpu_baseline(dict(inputs.CONFIGS[args.config]), args.cpu_states)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def oracle_sample(cfg, ns, nsteps, warm=0):
    """time `nsteps` steady ABM steps of the oracle on ns + ns states of the workload's lattice."""
    import numpy as np
    from oracle import ref
    from paper_2009_00745_b200 import inputs
    shape = tuple(cfg["shape"])
    both = cfg["nwf"][1] > 0
    nwf = (ns, ns if both else 0)
    oc = ref.RefContext(*shape, cfg["dx"], cfg["dt"], *nwf)
    for q in (0, 1):
        if nwf[q] == 0:
            continue
        psi = inputs.make_species(cfg, q, nwf[q], seed=inputs.SEED0).numpy()
        oc.set_wavefunctions(q, psi)
        z = np.zeros_like(psi)
        oc.set_history(q, psi, z, z, z, z)        # marks the multistep method as started: next steps are ABM steps
    cores = ref.set_num_threads(0)
    if warm:
        oc.step(warm)
    t0 = time.time()
    oc.step(nsteps)
    dt = time.time() - t0
    oc.close()
    return (nwf[0] + nwf[1]) * nsteps / dt, dt, cores, nwf


def cpu_baseline(cfg, ns):
    v, dt, cores, nwf = oracle_sample(cfg, ns, 1)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{nwf[0]}+{nwf[1]} states x 1 ABM step on the {cfg['name']} lattice ({dt:.1f} s), history pre-filled"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, nwf = workload(args.config, args.nwf)
    ns = args.cpu_states
    t0 = time.time()
    v, dt, cores, snwf = oracle_sample(cfg, ns, args.steps, warm=args.warmup)
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": cfg["name"], "lattice": list(cfg["shape"]), "dx_fm": cfg["dx"], "dt_fm_c": cfg["dt"],
                      "states_per_gpu": list(nwf), "sample_states": list(snwf)},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": f"{snwf[0]}+{snwf[1]} states per step, {args.steps} ABM steps after {args.warmup} warm-up"},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0, "wall_s": time.time() - t0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (default 1: the 24^3 workload)")
    ap.add_argument("--nwf", type=int, nargs=2, default=None, help="override states per species per GPU (testing)")
    ap.add_argument("--chunk", type=int, default=0, help="states per kernel launch (0 = the library's default)")
    ap.add_argument("--dgroup", type=int, default=0, help="chunks per density launch (0 = the library's default)")
    ap.add_argument("--also", type=int, nargs="*", default=[2],
                    help="further configs timed in the same invocation and reported under \"also\" (default: 2, the 32^3 workload)")
    ap.add_argument("--no-e2e", dest="e2e", action="store_false")
    ap.add_argument("--no-cpu-baseline", dest="cpu_baseline", action="store_false")
    ap.add_argument("--cpu-states", type=int, default=0, help="oracle sample: states per species (0 = sized from the host core count)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: warm-up raised to 3 (timing rules)", file=sys.stderr)
        args.warmup = 3
    if args.cpu_states <= 0:
        cores = os.cpu_count() or 4
        # the oracle costs about 0.5 core-seconds per qpwf-update on the 24^3 lattice: ~12 s for the
        # cpu_baseline sample, ~2 s per step for the reference arm (W + K steps)
        args.cpu_states = min(512, 12 * cores) if args.impl == "ours" else min(256, 2 * cores)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
