"""lise_renormalize_static, the one entry point of liblise.so that allocates nothing, against the existing path.

Why the entry point exists: a TDSLDA run fills the GPU with wavefunctions and their multistep history, usually out of the
application's own memory pool, so a caller in that position cannot let the library cudaMalloc (there is nothing left to
give, and a cudaMalloc / cudaFree pair stalls the whole device in the middle of a time loop).  Its per-state scratch is
a fixed array inside the library, shared by every call on a device and never cleared, so what this file checks is that
(1) it gives what the allocating path gives -- lise_params.renormalize = 1 inside lise_step, whose scratch belongs to a
context -- and (2) a second call right behind the first, with fewer states, is not disturbed by what the first left in
the array.  The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process (the first call does the per-device address lookup itself) and
after the other tests.
"""
import pytest
import torch

from paper_2009_00745_b200 import inputs
from tests.test_gpu_parity import TOL_WF

pytestmark = pytest.mark.gpu

SHAPE, NWF, SEED = (12, 8, 16), (20, 12), 41


def _stepped(renormalize):
    """one step of the library from off-norm states; returns y_1 of both species (CUDA tensors) and dV."""
    from paper_2009_00745_b200 import lise
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = SHAPE
    par = lise.default_params(); par.renormalize = int(renormalize)
    gc = lise.Lise(*SHAPE, cfg["dx"], cfg["dt"], *NWF, params=par)
    for q in (0, 1):
        psi = inputs.make_species(cfg, q, NWF[q], seed=SEED)
        # a different norm for every state (0.64 .. 1.7), so that a norm read from the wrong slot of the scratch shows
        scale = torch.linspace(0.8, 1.3, NWF[q], dtype=torch.float64).reshape(-1, 1, 1, 1, 1)
        gc.set_wavefunctions(q, (psi * scale).cuda())
    gc.step(1)      # the step ends with psi_k <- psi_k / |psi_k| when renormalize = 1 (lise.cu: starter_step)
    out = [gc.get_wavefunctions(q) for q in (0, 1)]
    gc.close()
    return out, cfg["dx"] ** 3


def _rel(a, b):
    return float((a - b).abs().max() / b.abs().max())


def test_static_renormalisation_matches_the_allocating_path_on_two_calls_in_a_row():
    from paper_2009_00745_b200 import lise
    want, dV = _stepped(renormalize=True)        # existing path: normalised inside lise_step
    got, _ = _stepped(renormalize=False)         # same step, left un-normalised ...
    norms_before = [dV * (g.abs() ** 2).sum(dim=(1, 2, 3, 4)) for g in got]
    assert float((norms_before[0] - 1).abs().min()) > 1e-3          # ... and really off norm
    torch.cuda.synchronize()
    # two calls back to back on one stream, no synchronisation between them: 20 states, then 12.  The second call finds
    # the 20 norms of the first still in the array; it must use only the 12 it writes itself.
    lise.renormalize_static(got[0], dV)
    free_before = torch.cuda.mem_get_info()[0]
    lise.renormalize_static(got[1], dV)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the amount of free device memory"
    for q in (0, 1):
        err = _rel(got[q], want[q])
        print(f"species {q}: static vs allocating renormalisation, max relative difference {err:.2e}")
        assert err < TOL_WF, (q, err)
        n = dV * (got[q].abs() ** 2).sum(dim=(1, 2, 3, 4))
        assert float((n - 1).abs().max()) < 1e-13, q
    # a third call on already normalised states changes nothing beyond round-off
    again = got[0].clone()
    lise.renormalize_static(again, dV)
    assert _rel(again, got[0]) < 1e-15


def test_static_renormalisation_refuses_more_states_than_its_scratch_holds():
    from paper_2009_00745_b200 import lise
    n = lise.STATIC_MAX_STATES + 1
    psi = torch.full((n, 2), 2.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(lise.LiseError, match="LISE_STATIC_MAX_STATES"):
        lise.renormalize_static(psi, 1.0)
    torch.cuda.synchronize()
    assert bool((psi == 2.0).all()), "a refused call must not touch the array"
    # the limit itself is accepted; zero states and an all-zero state are no-ops
    ok = psi[: lise.STATIC_MAX_STATES]
    ok[5] = 0.0
    lise.renormalize_static(ok, 0.5)
    lise.renormalize_static(psi[:0], 0.5)
    torch.cuda.synchronize()
    norms = 0.5 * (ok.abs() ** 2).sum(dim=1)
    assert float(norms[5]) == 0.0 and bool(torch.isfinite(ok.real).all())
    keep = torch.ones(lise.STATIC_MAX_STATES, dtype=torch.bool, device="cuda"); keep[5] = False
    assert float((norms[keep] - 1).abs().max()) < 1e-14
