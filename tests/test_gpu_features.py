"""GPU parity of the "next" features against the CPU oracle, through the C-ABI binding, on the same
seeded inputs: restart, renormalisation, observables of Eqs. 37-41, functional variants (Eqs. 8, 10, 15, 20), boosts,
external fields and frame terms (Eqs. 23-36).  Tolerances are north_star's (wavefunctions 1e-10, densities 1e-11,
energy 1e-10); potentials 1e-10 as in test_gpu_parity.py.
"""
import numpy as np
import pytest
import torch

from oracle import ref
from paper_2009_00745_b200 import inputs
from tests.test_gpu_parity import TOL_DENS, TOL_E, TOL_WF, field_rel, rel

pytestmark = pytest.mark.gpu


def _copy_params(src, dst):
    for name, _ in src._fields_:
        v = getattr(src, name)
        if hasattr(v, "__len__"):
            getattr(dst, name)[:] = list(v)
        else:
            setattr(dst, name, v)
    return dst


def _pair(shape, nwf, seed, edit=None, dt=0.05, cfg_idx=1):
    """(cfg, psi, oracle ctx, gpu ctx) with the same parameters; edit(params) modifies the defaults."""
    from paper_2009_00745_b200 import lise
    cfg = dict(inputs.CONFIGS[cfg_idx]); cfg["shape"] = shape
    psi = [inputs.make_species(cfg, q, nwf[q], seed=seed) for q in (0, 1)]
    po = ref.default_params()
    if nwf[1] == 0:
        po.coulomb = 0
    if edit:
        edit(po)
    pg = _copy_params(po, lise.default_params())
    oc = ref.RefContext(*shape, cfg["dx"], dt, *nwf, params=po)
    gc = lise.Lise(*shape, cfg["dx"], dt, *nwf, params=pg)
    for q in (0, 1):
        oc.set_wavefunctions(q, psi[q].numpy())
        gc.set_wavefunctions(q, psi[q].cuda())
    return cfg, psi, oc, gc


def _compare_state(oc, gc, nwf, what):
    for q in (0, 1):
        if nwf[q] == 0:
            continue
        assert rel(gc.get_wavefunctions(q).cpu().numpy(), oc.get_wavefunctions(q)) < TOL_WF, (what, "wavefunctions", q)
        assert field_rel(gc.densities(q).cpu().numpy(), oc.densities(q)) < TOL_DENS, (what, "densities", q)
        assert field_rel(gc.potentials(q).cpu().numpy(), oc.potentials(q)) < 1e-10, (what, "potentials", q)
    eo, eg = oc.observables(), gc.observables()
    assert abs(eg["energy"] - eo["energy"]) < TOL_E * abs(eo["energy"]), (what, eg, eo)
    assert eg["step"] == eo["step"] and abs(eg["time"] - eo["time"]) < 1e-12


def _compare_ext(oc, gc, what):
    a, b = oc.observables_ext(), gc.observables_ext()
    scale = {"rcm": 1.0, "rcm_n": 1.0, "rcm_p": 1.0, "v_cm": 1e-3}
    for k, v in a.items():
        va, vb = np.atleast_1d(v), np.atleast_1d(b[k])
        ref_scale = max(np.abs(va).max(), scale.get(k, 0.0))
        if k in ("q20", "q30", "q40", "q21", "q22"):
            ref_scale = max(ref_scale, 1e-6 * abs(a["q40"]) ** (int(k[1]) / 4.0), 1.0)
        assert np.abs(va - vb).max() <= 1e-9 * max(ref_scale, 1e-12), (what, k, va, vb)


def test_restart_through_the_starter():
    """L764-L768: download y_n, new context, upload (history reset), set the clock, continue: the same on both sides."""
    from paper_2009_00745_b200 import lise
    shape, nwf = (16, 16, 16), (14, 10)
    cfg, psi, oc, gc = _pair(shape, nwf, seed=31)
    oc.step(5); gc.step(5)
    t5 = gc.observables()["time"]
    host = [torch.empty((nwf[q], 4) + shape, dtype=torch.complex128) for q in (0, 1)]
    for q in (0, 1):
        gc.download_wavefunctions(q, host[q])
    y5 = [oc.get_wavefunctions(q) for q in (0, 1)]
    gc.close(); oc.close()
    oc2 = ref.RefContext(*shape, cfg["dx"], 0.05, *nwf)
    gc2 = lise.Lise(*shape, cfg["dx"], 0.05, *nwf)
    for q in (0, 1):
        oc2.set_wavefunctions(q, y5[q])
        gc2.upload_wavefunctions(q, host[q])
    oc2.set_time(t5, 5); gc2.set_time(t5, 5)
    oc2.step(4); gc2.step(4)                                        # 3 starter steps + 1 ABM step
    _compare_state(oc2, gc2, nwf, "restart")
    assert gc2.observables()["step"] == 9
    gc2.close(); oc2.close()


def test_renormalisation_every_step():
    """L637 (lise_params.renormalize): off-norm input, 3 starter + 3 ABM steps."""
    def edit(p):
        p.renormalize = 1
    shape, nwf = (12, 8, 16), (9, 7)
    cfg, psi, oc, gc = _pair(shape, nwf, seed=32, edit=edit, cfg_idx=0)
    for q in (0, 1):
        oc.set_wavefunctions(q, 1.002 * psi[q].numpy()); gc.set_wavefunctions(q, (1.002 * psi[q]).cuda())
    gc.set_chunk(4)
    oc.step(6); gc.step(6)
    _compare_state(oc, gc, nwf, "renormalize")
    assert gc.observables()["norm_defect"] < 1e-14
    gc.close(); oc.close()


def test_observables_of_eqs_37_to_41():
    shape, nwf = (16, 16, 16), (12, 9)
    cfg, psi, oc, gc = _pair(shape, nwf, seed=33)
    _compare_ext(oc, gc, "initial")
    oc.step(4); gc.step(4)
    _compare_ext(oc, gc, "after 4 steps")
    gc.close(); oc.close()


def _seall1(p):
    p.functional = 1
    p.sea_a[:] = (-62.0, 30.0, -9.0); p.sea_b[:] = (-410.0, 160.0, 40.0); p.sea_c[:] = (520.0, -90.0, 25.0)
    p.sea_cdn[:] = (-58.0, 14.0); p.sea_cdj[:] = (-73.0, -27.0)


def _surface_pairing(p):
    p.alpha_pair = 0.5


def _spherical_cutoff(p):
    p.pairing_cutoff = 1; p.mu_n = -6.0; p.mu_p = -4.0; p.e_cut = 55.0; p.alpha_pair = 1.0


@pytest.mark.parametrize("edit", [_seall1, _surface_pairing, _spherical_cutoff], ids=["seall1", "mixed_pairing", "eq20_cutoff"])
def test_functional_variants(edit):
    """Eqs. 10 / 15 (SeaLL1 form with caller-supplied coefficients), Eq. 8 (alpha != 0), Eq. 20 (spherical cutoff)."""
    shape, nwf = (12, 12, 12), (10, 8)
    cfg, psi, oc, gc = _pair(shape, nwf, seed=34, edit=edit, cfg_idx=0)
    _compare_state(oc, gc, nwf, "initial")
    oc.step(5); gc.step(5)
    _compare_state(oc, gc, nwf, "after 5 steps")
    gc.close(); oc.close()


def test_boost_external_fields_and_frames():
    """Eq. 23 boost, Eq. 24 scalar + vector fields, Eq. 26 c.m. velocity, Eq. 36 rotating frame: potentials (U, A, S),
    H psi, the energy of the external terms and 5 time steps."""
    shape, nwf = (16, 12, 8), (8, 6)
    cfg, psi, oc, gc = _pair(shape, nwf, seed=35, cfg_idx=0)
    rng = np.random.default_rng(36)
    x = np.meshgrid(*[np.arange(n) * cfg["dx"] for n in shape], indexing="ij")
    L = [n * cfg["dx"] for n in shape]
    chi = 0.3 * np.sin(2 * np.pi * x[0] / L[0]) + 2 * np.pi * x[2] / L[2]
    for q in (0, 1):
        u0 = 2.0 * np.cos(2 * np.pi * x[1] / L[1]) * (1 + q)
        uv = 0.01 * np.stack([np.sin(2 * np.pi * x[(i + 1) % 3] / L[(i + 1) % 3] + q) for i in range(3)])
        oc.set_external_fields(q, u0=u0, uvec=uv)
        gc.set_external_fields(q, u0=torch.from_numpy(u0).cuda(), uvec=torch.from_numpy(np.ascontiguousarray(uv)).cuda())
        oc.boost(q, chi); gc.boost(q, torch.from_numpy(np.ascontiguousarray(chi)).cuda())
    frame = dict(v_cm=(0.004, -0.002, 0.006), omega=(0.0004, -0.0003, 0.0007), origin=(0.5 * L[0], 0.5 * L[1], 0.4 * L[2]))
    oc.set_frame(**frame); gc.set_frame(**frame)
    _compare_state(oc, gc, nwf, "initial")
    for q in (0, 1):
        probe = inputs.make_species(cfg, q, 3, seed=37)
        h_ref = oc.apply_h(q, probe.numpy()).reshape(probe.shape)
        assert rel(gc.apply_h(q, probe.cuda()).cpu().numpy(), h_ref) < 1e-12, ("H psi", q)
    _compare_ext(oc, gc, "external terms")
    oc.step(5); gc.step(5)
    _compare_state(oc, gc, nwf, "after 5 steps")
    # switching everything off again restores the plain potentials
    for q in (0, 1):
        oc.set_external_fields(q); gc.set_external_fields(q)
    oc.set_frame(); gc.set_frame()
    for q in (0, 1):
        assert field_rel(gc.potentials(q).cpu().numpy(), oc.potentials(q)) < 1e-10
    gc.close(); oc.close()


def test_driven_external_fields_with_amplitude_pairs():
    """U0(r) f(t), Uvec(r) f(t) with (f(t_n), f(t_{n+1})) set before every step: 3 starter + 4 ABM steps,
    potentials and e_ext at an amplitude other than 1, against the oracle (whose driven stepping is pinned to the closed
    form of a driven free state)."""
    shape, nwf = (12, 12, 16), (8, 6)
    cfg, psi, oc, gc = _pair(shape, nwf, seed=38, cfg_idx=0)
    x = np.meshgrid(*[np.arange(n) * cfg["dx"] for n in shape], indexing="ij")
    L = [n * cfg["dx"] for n in shape]
    for q in (0, 1):
        u0 = 6.0 * np.cos(2 * np.pi * x[2] / L[2]) * (1 + q) + 3.0
        uv = 0.01 * np.stack([np.cos(2 * np.pi * x[(i + 2) % 3] / L[(i + 2) % 3] + q) for i in range(3)])
        oc.set_external_fields(q, u0=u0, uvec=uv)
        gc.set_external_fields(q, u0=torch.from_numpy(u0).cuda(), uvec=torch.from_numpy(np.ascontiguousarray(uv)).cuda())
    f = lambda t: np.cos(2.0 * t) + 0.5 * t
    dt = cfg["dt"]
    for i in range(7):
        for c in (oc, gc):
            c.set_external_amplitudes(f(i * dt), f((i + 1) * dt))
            c.step(1)
    for c in (oc, gc):
        c.set_external_amplitudes(f(7 * dt), f(8 * dt))
    _compare_state(oc, gc, nwf, "driven, after 7 steps")
    _compare_ext(oc, gc, "driven external terms")
    # the run really was driven: a static field (amplitudes 1, 1 throughout) ends elsewhere
    cfg2, psi2, oc2, gc2 = _pair(shape, nwf, seed=38, cfg_idx=0)
    oc2.close()
    for q in (0, 1):
        u0 = 6.0 * np.cos(2 * np.pi * x[2] / L[2]) * (1 + q) + 3.0
        gc2.set_external_fields(q, u0=torch.from_numpy(u0).cuda())
    gc2.step(7)
    assert rel(gc2.get_wavefunctions(0).cpu().numpy(), gc.get_wavefunctions(0).cpu().numpy()) > 1e-6
    gc2.close(); gc.close(); oc.close()


def test_static_solution_stays_stationary_on_the_gpu():
    """A self-consistent Hartree-Fock state (built on the CPU by dense diagonalisation in the oracle's mean field,
    tests/dense_ref.py; pairing off, Coulomb on, 2 + 2 particles on 8^3: the FFT H-apply kernels) is a fixed point of the
    phase-removed evolution (Eqs. 80-81): after 3 starter + 7 ABM steps of the CUDA path wavefunctions, density and
    energy are those of the input, and H psi_k = -eps_k psi_k for the occupied v-type states."""
    from paper_2009_00745_b200 import lise
    from tests import dense_ref
    shape, a, dt = (8, 8, 8), 1.5, 0.05
    po = ref.default_params(); po.g0_n = 0.0; po.g0_p = 0.0
    oc = ref.RefContext(*shape, a, dt, 2, 2, params=po)
    psi, eps, it, change = dense_ref.scf_ground_state(oc, shape, a)
    assert change < 1e-13, (it, change)
    pg = _copy_params(po, lise.default_params())
    gc = lise.Lise(*shape, a, dt, 2, 2, params=pg)
    dev = [torch.from_numpy(p).cuda() for p in psi]
    for q in (0, 1):
        gc.set_wavefunctions(q, dev[q])
    o0 = gc.observables()
    d0 = [gc.densities(q).cpu().numpy() for q in (0, 1)]
    for q in (0, 1):
        hp = gc.apply_h(q, dev[q]).cpu().numpy()
        for k in range(2):
            assert np.abs(hp[k] + eps[q][k] * psi[q][k]).max() < 1e-9 * abs(eps[q][k]) * np.abs(psi[q][k]).max() + 1e-11
    gc.step(10)
    o1 = gc.observables()
    for q in (0, 1):
        got = gc.get_wavefunctions(q).cpu().numpy()
        assert np.abs(got - psi[q]).max() < 1e-11 * np.abs(psi[q]).max()
        d1 = gc.densities(q).cpu().numpy()
        assert np.abs(d1[0] - d0[q][0]).max() < 1e-12 * np.abs(d0[q][0]).max()
    assert abs(o1["energy"] - o0["energy"]) < 1e-12 * abs(o0["energy"])
    assert abs(o1["n_neutron"] - 2.0) < 1e-12 and abs(o1["n_proton"] - 2.0) < 1e-12
    gc.close(); oc.close()
