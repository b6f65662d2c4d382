"""Pins of the CPU oracle against what PAPER.md and the mathematics fix (CPU only, no CUDA).

Each test names the passage it pins and the plausible mistake it would catch.
"""
import json
import math
import os

import numpy as np
import pytest
import scipy.integrate
import scipy.special

from oracle import ref
from tests import dense_ref as dr

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.json")))


def rel(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


# ---------------------------------------------------------------------------------------------
# constants printed by the paper
# ---------------------------------------------------------------------------------------------
def test_pairing_constant_K_matches_printed_value_and_integral():
    """Eq. 21 / L211: K printed to 16 digits, and defined by an integral."""
    val, _ = scipy.integrate.quad(lambda t: math.log(1.0 + 1.0 / math.cos(t) ** 2), 0.0, math.pi / 4,
                                  epsabs=1e-15, epsrel=1e-15)
    assert abs(12.0 / math.pi * val - GOLD["pairing_K"]["value"]) < 2e-15
    assert ref.pairing_K() == GOLD["pairing_K"]["value"]


def test_pde_count_printed_by_paper():
    """L651: 16 Nx Ny Nz PDEs = 2 species x 2 Nxyz states x 4 components."""
    for lat, cnt in zip(GOLD["pde_counts"]["lattices"], GOLD["pde_counts"]["counts"]):
        assert 2 * (2 * lat[0] * lat[1] * lat[2]) * 4 == cnt


# ---------------------------------------------------------------------------------------------
# lattice derivatives (Eqs. 43-50, 48)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [6, 12, 24, 32, 40, 64])
def test_derivative_matrices_equal_dvr_closed_forms(N):
    """Eq. 48a and (corrected) Eq. 48b equal F^-1 (ik)^m F built from Eq. 49 sums."""
    a = 1.25
    c = ref.RefContext(N, 4, 4, a, 0.05, 0, 0)
    d1, d2 = c.deriv_matrix(0, 1), c.deriv_matrix(0, 2)
    assert np.abs(d1 - dr.dvr_d1(N, a)).max() < 2e-14 * np.pi / a
    assert np.abs(d2 - dr.dvr_d2(N, a)).max() < 2e-14 * (np.pi / a) ** 2
    # the printed prefactor pi^2/(2 N^2 a^2) of Eq. 48b fails the zero-row-sum property of a derivative
    assert abs(d2.sum(axis=1)).max() < 1e-12
    assert abs(d1 + d1.T).max() < 1e-14 and abs(d2 - d2.T).max() < 1e-13


def test_plane_wave_derivatives_exact_incl_nyquist():
    """L412: derivatives of lattice plane waves are exact; odd order is zeroed at the Nyquist mode."""
    shape, a = (12, 24, 32), 1.1
    c = ref.RefContext(*shape, a, 0.05, 0, 0)
    x = [np.arange(n) * a for n in shape]
    X = np.meshgrid(*x, indexing="ij")
    for modes in [(1, 2, 3), (5, -7, 11), (6, 12, 16), (-3, 0, 15)]:
        k = [2 * np.pi * m / (n * a) for m, n in zip(modes, shape)]
        f = np.exp(1j * sum(ki * Xi for ki, Xi in zip(k, X)))
        for ax in range(3):
            nyq = abs(modes[ax]) * 2 == shape[ax]
            d1 = c.deriv(ax, 1, f)
            d2 = c.deriv(ax, 2, f)
            want1 = 0 * f if nyq else 1j * k[ax] * f
            assert np.abs(d1 - want1).max() < 5e-13
            assert np.abs(d2 + k[ax] ** 2 * f).max() < 5e-12


def test_derivative_equals_library_fft_on_random_field():
    """special case that reduces to a library routine: numpy.fft along one axis."""
    shape, a = (24, 12, 40), 1.25
    rng = np.random.default_rng(7)
    f = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    c = ref.RefContext(*shape, a, 0.05, 0, 0)
    for ax in range(3):
        n = shape[ax]
        k = 2 * np.pi * np.fft.fftfreq(n, d=a)
        k1 = k.copy(); k1[n // 2] = 0.0
        sh = [1, 1, 1]; sh[ax] = n
        fk = np.fft.fft(f, axis=ax)
        w1 = np.fft.ifft(1j * k1.reshape(sh) * fk, axis=ax)
        w2 = np.fft.ifft(-(k ** 2).reshape(sh) * fk, axis=ax)
        assert rel(c.deriv(ax, 1, f), w1) < 1e-13
        assert rel(c.deriv(ax, 2, f), w2) < 1e-13


# ---------------------------------------------------------------------------------------------
# H-apply against the brute-force dense matrix (Eqs. 11, 12, 55, 56)
# ---------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def dense_case():
    shape, a = (6, 4, 6), 1.25
    rng = np.random.default_rng(11)
    pot = dr.random_potentials(shape, rng)
    L = sum(dr.kron3(dr.dvr_d2(shape[i], a), shape, i) for i in range(3))
    H = dr.dense_H(shape, a, pot)
    c = ref.RefContext(*shape, a, 0.05, 0, 0)
    return shape, a, pot, dr.table3(pot, L @ pot["M"], shape), H, c, rng


def test_apply_h_equals_dense_matrix(dense_case):
    """every term of Eq. 12 (signs, spin structure, symmetrisations) and the block structure of Eq. 11."""
    shape, a, pot, t3, H, c, rng = dense_case
    nxyz = int(np.prod(shape))
    psi = rng.standard_normal((5, 4 * nxyz)) + 1j * rng.standard_normal((5, 4 * nxyz))
    got = c.apply_h_with(t3, psi).reshape(5, -1)
    want = psi @ H.T
    assert np.abs(got - want).max() < 1e-12 * np.abs(want).max()


def test_dense_H_is_hermitian_and_spectrum_symmetric(dense_case):
    """Eq. 11: H Hermitian, eigenvalues come in +-E pairs."""
    shape, a, pot, t3, H, c, rng = dense_case
    assert np.abs(H - H.conj().T).max() < 1e-12 * np.abs(H).max()
    ev = np.linalg.eigvalsh(H)
    assert np.abs(ev + ev[::-1]).max() < 1e-10 * np.abs(ev).max()


def test_oracle_h_hermitian_on_random_vectors():
    """<a|Hb> = <Ha|b> on a bigger non-cubic lattice with non-smooth potentials."""
    shape, a = (12, 6, 8), 1.0
    rng = np.random.default_rng(5)
    pot = dr.random_potentials(shape, rng, smooth=False)
    c = ref.RefContext(*shape, a, 0.05, 0, 0)
    lapM = sum(c.deriv(i, 2, pot["M"].reshape(shape).astype(complex)).real for i in range(3))
    t3 = dr.table3(pot, lapM.reshape(-1), shape)
    n = 4 * int(np.prod(shape))
    x = rng.standard_normal((2, n)) + 1j * rng.standard_normal((2, n))
    hx = c.apply_h_with(t3, x).reshape(2, n)
    lhs = np.vdot(x[0], hx[1]); rhs = np.vdot(hx[0], x[1])
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    assert abs(np.vdot(x[0], hx[0]).imag) < 1e-12 * abs(np.vdot(x[0], hx[0]))


# ---------------------------------------------------------------------------------------------
# densities, potentials, energy: variational identity H = dE/d psi^dagger (L643)
# ---------------------------------------------------------------------------------------------
def _smooth_states(shape, a, nst, rng, kc=1.0):
    k = np.meshgrid(*[2 * np.pi * np.fft.fftfreq(n, d=a) for n in shape], indexing="ij")
    mask = sum(q * q for q in k) < kc * kc
    psi = np.zeros((nst, 4) + tuple(shape), complex)
    for s in range(nst):
        for cpt in range(4):
            co = (rng.uniform(-1, 1, shape) + 1j * rng.uniform(-1, 1, shape)) * mask
            psi[s, cpt] = np.fft.ifftn(co) * (0.3 if cpt >= 2 else 0.9)
    dV = a ** 3
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2, 3, 4), keepdims=True) * dV)
    return psi


def _energy(c, psi_n, psi_p):
    dn = c.densities_of(psi_n) if psi_n is not None and len(psi_n) else np.zeros((14,) + c.shape)
    dp = c.densities_of(psi_p) if psi_p is not None and len(psi_p) else np.zeros((14,) + c.shape)
    pn, pp, e5 = c.potentials_from(dn, dp)
    return e5, pn, pp, dn, dp


def test_energy_gradient_equals_h_pairing_off():
    """finite-difference dE along arbitrary directions g of the v components equals 2 Re<h* v|g>,
    i.e. -(H psi)_v: pins U (incl. the terms missing from Eq. 14), M, W, S, A signs and xi factors,
    the spin density convention, tau via Eq. 51, div J, Coulomb direct + exchange."""
    shape, a = (8, 6, 10), 1.25
    rng = np.random.default_rng(3)
    c = ref.RefContext(*shape, a, 0.05, 3, 2)
    par = ref.default_params(); par.g0_n = 0.0; par.g0_p = 0.0; par.coulomb = 1
    c.set_params(par)
    psi = [_smooth_states(shape, a, 3, rng), _smooth_states(shape, a, 2, rng)]
    # scale v up so that densities are nuclear-sized (n ~ 0.1 fm^-3)
    for p in psi:
        p[:, 2:] *= 6.0
    e5, pn, pp, dn, dp = _energy(c, psi[0], psi[1])
    pots = [pn, pp]
    dV = a ** 3
    for q in (0, 1):
        hpsi = c.apply_h_with(pots[q], psi[q]).reshape(psi[q].shape)
        for trial in range(2):
            g = np.zeros_like(psi[q])
            g[:, 2:] = _smooth_states(shape, a, len(psi[q]), rng)[:, 2:]
            want = 2.0 * np.real(np.vdot(-hpsi[:, 2:], g[:, 2:])) * dV
            h = 1e-5
            trial_p = [p.copy() for p in psi]; trial_m = [p.copy() for p in psi]
            trial_p[q] = psi[q] + h * g; trial_m[q] = psi[q] - h * g
            ep = _energy(c, *trial_p)[0][0]; em = _energy(c, *trial_m)[0][0]
            fd = (ep - em) / (2 * h)
            assert abs(fd - want) < 2e-7 * max(abs(want), 1.0), (q, fd, want)


def test_energy_stationary_along_flow_pairing_off():
    """dE/dt = 0 along f = -i H psi / (hbar c) for ARBITRARY states when pairing is off (L643)."""
    shape, a = (8, 8, 6), 1.25
    rng = np.random.default_rng(8)
    c = ref.RefContext(*shape, a, 0.05, 4, 3)
    par = ref.default_params(); par.g0_n = 0.0; par.g0_p = 0.0
    c.set_params(par)
    psi = [_smooth_states(shape, a, 4, rng), _smooth_states(shape, a, 3, rng)]
    for p in psi:
        p[:, 2:] *= 5.0
    e5, pn, pp, dn, dp = _energy(c, *psi)
    f = [c.apply_h_with(pot, p).reshape(p.shape) / (1j * par.hbarc) for pot, p in zip((pn, pp), psi)]
    scale = sum(np.sqrt((np.abs(x) ** 2).sum()) for x in f)
    h = 1e-4 / scale
    ep = _energy(c, psi[0] + h * f[0], psi[1] + h * f[1])[0][0]
    em = _energy(c, psi[0] - h * f[0], psi[1] - h * f[1])[0][0]
    # compare with the size of the same derivative along a generic direction
    g = [_smooth_states(shape, a, len(p), rng) for p in psi]
    gp = _energy(c, psi[0] + h * scale * g[0], psi[1] + h * scale * g[1])[0][0]
    gm = _energy(c, psi[0] - h * scale * g[0], psi[1] - h * scale * g[1])[0][0]
    assert abs(ep - em) < 1e-6 * abs(gp - gm)


def test_galilean_boost_energy():
    """Eq. 23 boost with a lattice wavevector q: E' - E = (hbar^2/2m)(q^2 N + 2 q . int j)
    (pins the signs of the time-odd terms A, S and of j; L179)."""
    shape, a = (8, 8, 10), 1.25
    rng = np.random.default_rng(21)
    c = ref.RefContext(*shape, a, 0.05, 3, 3)
    par = ref.default_params()
    c.set_params(par)
    psi = [_smooth_states(shape, a, 3, rng, kc=0.9), _smooth_states(shape, a, 3, rng, kc=0.9)]
    for p in psi:
        p[:, 2:] *= 5.0
    e0, _, _, dn, dp = _energy(c, *psi)
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    qv = [2 * np.pi * m / (n * a) for m, n in zip((1, 0, -1), shape)]
    ph = np.exp(1j * sum(qi * xi for qi, xi in zip(qv, x)))
    boosted = []
    for p in psi:
        b = p.copy(); b[:, :2] *= ph; b[:, 2:] *= np.conj(ph)
        boosted.append(b)
    e1 = _energy(c, *boosted)[0]
    dV = a ** 3
    N = (dn[0].sum() + dp[0].sum()) * dV
    qj = sum(qv[i] * (dn[6 + i].sum() + dp[6 + i].sum()) for i in range(3)) * dV
    want = par.hbar2_2m * (sum(q * q for q in qv) * N + 2 * qj)
    assert abs((e1[0] - e0[0]) - want) < 1e-9 * abs(e0[0])
    # pairing energy is invariant (kappa only picks up a phase)
    assert abs(e1[4] - e0[4]) < 1e-10 * abs(e0[4])


def test_kinetic_energy_consistent_with_tau():
    """sum_k <phi_k|T|phi_k> = dV sum M tau with T of Eq. 55 and tau of Eq. 51 (reading B11)."""
    shape, a = (8, 6, 8), 1.25
    rng = np.random.default_rng(2)
    c = ref.RefContext(*shape, a, 0.05, 4, 0)
    psi = _smooth_states(shape, a, 4, rng)
    pot = dr.random_potentials(shape, rng)
    for key in ("W", "S", "A"):
        pot[key] = [0 * f for f in pot[key]]
    pot["U"] = 0 * pot["U"]; pot["Delta"] = 0 * pot["Delta"]
    lapM = sum(c.deriv(i, 2, pot["M"].reshape(shape).astype(complex)).real for i in range(3))
    t3 = dr.table3(pot, lapM.reshape(-1), shape)
    hpsi = c.apply_h_with(t3, psi).reshape(psi.shape)
    # (H psi)_v = -conj(h conj v)  =>  <phi|T|phi> = -Re <v|(H psi)_v>
    lhs = -np.real(np.vdot(psi[:, 2:], hpsi[:, 2:]))
    dens = c.densities_of(psi)
    rhs = (pot["M"].reshape(shape) * dens[1]).sum()
    assert abs(lhs - rhs) < 1e-11 * abs(rhs)


def test_density_definitions_on_single_plane_wave_state():
    """closed forms for one state v_up = A e^{ik.r}, v_dn = B e^{ik'.r}, u_up = C e^{ip.r}:
    n, tau (Eq. 3c value), j (Eq. 3f), s (Eq. 3d with phi = v*), kappa (Eq. 3b)."""
    shape, a = (8, 8, 8), 1.0
    c = ref.RefContext(*shape, a, 0.05, 1, 0)
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    L = 8 * a
    k = 2 * np.pi / L * np.array([1, 2, -1]); kp = 2 * np.pi / L * np.array([-2, 1, 3]); p = 2 * np.pi / L * np.array([0, 1, 1])
    A, B, Cc = 0.3 + 0.1j, -0.2 + 0.25j, 0.5 - 0.4j
    pw = lambda q: np.exp(1j * sum(qi * xi for qi, xi in zip(q, x)))
    psi = np.zeros((1, 4) + shape, complex)
    psi[0, 0] = Cc * pw(p); psi[0, 2] = A * pw(k); psi[0, 3] = B * pw(kp)
    d = c.densities_of(psi)
    n = abs(A) ** 2 + abs(B) ** 2
    assert np.abs(d[0] - n).max() < 1e-13
    # tau = |grad v|^2 for plane waves (Eq. 3c), reached through Eq. 51
    assert np.abs(d[1] - (abs(A) ** 2 * k @ k + abs(B) ** 2 * kp @ kp)).max() < 1e-11
    # j = -Im(v^* grad v) summed = -(|A|^2 k + |B|^2 k')   (Eq. 3f)
    for i in range(3):
        assert np.abs(d[6 + i] + (abs(A) ** 2 * k[i] + abs(B) ** 2 * kp[i])).max() < 1e-12
    # s = phi^dagger sigma phi, phi = conj(v): phi_up^* phi_dn = v_up conj(v_dn)
    z = psi[0, 2] * np.conj(psi[0, 3])
    assert np.abs(d[2] - 2 * z.real).max() < 1e-13 and np.abs(d[3] - 2 * z.imag).max() < 1e-13
    assert np.abs(d[4] - (abs(A) ** 2 - abs(B) ** 2)).max() < 1e-13
    # kappa = conj(v_dn) u_up
    kap = np.conj(psi[0, 3]) * psi[0, 0]
    assert np.abs(d[12] - kap.real).max() < 1e-13 and np.abs(d[13] - kap.imag).max() < 1e-13
    # curl j of a uniform current vanishes; div J of this state: J_k = eps_kij Im(phi^+ sigma_j D_i phi)
    assert np.abs(d[9:12]).max() < 1e-11


# ---------------------------------------------------------------------------------------------
# pairing block, kappa convention, rearrangement term: particle-hole complete set
# ---------------------------------------------------------------------------------------------
def test_complete_set_conserves_energy_and_number_with_pairing():
    """all positive-energy eigenvectors of an Eq.-11 matrix on 4^3: kappa antisymmetric,
    dE/dt = dN/dt = 0 with pairing ON (needs the pairing rearrangement term in U)."""
    shape, a = (4, 4, 4), 1.5
    nxyz = 64
    rng = np.random.default_rng(17)
    pot = dr.random_potentials(shape, rng)
    pot["U"] = pot["U"] - 20.0
    H = dr.dense_H(shape, a, pot)
    ev, vec = np.linalg.eigh(H)
    pos = vec[:, ev > 0].T                      # rows = states, (u_up, u_dn, v_up, v_dn) x space
    assert pos.shape[0] == 2 * nxyz
    psi = pos.reshape(2 * nxyz, 4, *shape) / np.sqrt(a ** 3)
    c = ref.RefContext(*shape, a, 0.05, 2 * nxyz, 0)
    par = ref.default_params(); par.coulomb = 0
    c.set_params(par)
    d = c.densities_of(psi)
    # kappa = sum v_dn^* u_up = - sum v_up^* u_dn
    alt = (np.conj(psi[:, 2]) * psi[:, 1]).sum(axis=0)
    assert np.abs((d[12] + 1j * d[13]) + alt).max() < 1e-12 * np.abs(alt).max()

    def flow(rearr):
        par.pairing_rearrangement = rearr
        c.set_params(par)
        zero = np.zeros_like(d)
        pn, pp, e5 = c.potentials_from(d, zero)
        f = c.apply_h_with(pn, psi).reshape(psi.shape) / (1j * par.hbarc)
        h = 1e-4
        out = []
        for sgn in (+1, -1):
            dd = c.densities_of(psi + sgn * h * f)
            e = c.potentials_from(dd, zero)[2][0]
            out.append((e, dd[0].sum() * a ** 3))
        return (out[0][0] - out[1][0]) / (2 * h), (out[0][1] - out[1][1]) / (2 * h), e5[0]

    dE, dN, E = flow(1)
    assert abs(dN) < 1e-9
    assert abs(dE) < 1e-7 * abs(E)
    dE_no, _, _ = flow(0)
    assert abs(dE_no) > 20 * abs(dE)           # without the rearrangement term energy is not conserved


# ---------------------------------------------------------------------------------------------
# Coulomb (Eqs. 57-62)
# ---------------------------------------------------------------------------------------------
def test_coulomb_gaussian_closed_form():
    """isolated Gaussian charge: Phi = e^2 Q erf(r / (sqrt2 sigma)) / r, no periodic images."""
    shape, a, sig = (32, 32, 32), 1.0, 2.4
    c = ref.RefContext(*shape, a, 0.05, 0, 0)
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    ctr = [15.7 * a, 16.0 * a, 16.4 * a]
    r2 = sum((xi - ci) ** 2 for xi, ci in zip(x, ctr))
    Q = 20.0
    rho = Q * np.exp(-r2 / (2 * sig * sig)) / (2 * np.pi * sig * sig) ** 1.5
    phi = c.coulomb(rho)
    r = np.sqrt(r2)
    e2 = ref.default_params().e2
    want = e2 * Q * scipy.special.erf(r / (math.sqrt(2) * sig)) / np.where(r > 0, r, 1.0)
    assert np.abs(phi - want).max() < 1e-8 * np.abs(want).max()


def test_coulomb_noncubic_point_charges_by_direct_sum():
    """brute force on a tiny non-cubic lattice: Phi(r) = e^2 dV sum_r' n(r') f(r - r') with the
    lattice Green's function of the truncated kernel evaluated by explicit k-sums (Eq. 62)."""
    shape, a = (4, 6, 8), 1.0
    c = ref.RefContext(*shape, a, 0.05, 0, 0)
    rng = np.random.default_rng(4)
    rho = rng.uniform(0, 1, shape)
    phi = c.coulomb(rho)
    P = 3 * max(shape); D = math.sqrt(3) * a * max(shape)
    kk = 2 * np.pi * np.fft.fftfreq(P, d=a)
    K = np.meshgrid(kk, kk, kk, indexing="ij")
    k2 = sum(q * q for q in K)
    ft = np.where(k2 > 0, 4 * np.pi * (1 - np.cos(np.sqrt(k2) * D)) / np.where(k2 > 0, k2, 1), 2 * np.pi * D * D)
    pad = np.zeros((P, P, P)); pad[:shape[0], :shape[1], :shape[2]] = rho
    want = ref.default_params().e2 * np.real(np.fft.ifftn(np.fft.fftn(pad) * ft))[:shape[0], :shape[1], :shape[2]]
    assert rel(phi, want) < 1e-12


# ---------------------------------------------------------------------------------------------
# Adams-Bashforth-Milne (Eq. 78)
# ---------------------------------------------------------------------------------------------
def _poly_history(deg, dt, tn):
    y = lambda t: t ** deg
    f = lambda t: deg * t ** (deg - 1) if deg > 0 else 0.0 * t
    arr = lambda v: np.array([v], dtype=complex)
    return y, f, arr


@pytest.mark.parametrize("deg", [0, 1, 2, 3, 4])
def test_abm_exact_for_polynomials_up_to_degree_4(deg):
    """Eq. 78a with the restored coefficient 119 and Eq. 78c are exact for degree <= 4."""
    dt, tn = 0.37, 1.3
    y, f, arr = _poly_history(deg, dt, tn)
    p, m = ref.abm_predict(dt, arr(y(tn)), arr(y(tn - dt)), arr(f(tn)), arr(f(tn - dt)), arr(f(tn - 2 * dt)),
                           arr(f(tn - 3 * dt)), arr(0.0))
    assert abs(p[0] - y(tn + dt)) < 1e-13 * max(1, abs(y(tn + dt)))
    ynew, e = ref.abm_correct(dt, arr(y(tn)), arr(y(tn - dt)), arr(f(tn + dt)), arr(f(tn)), arr(f(tn - dt)),
                              arr(f(tn - 2 * dt)), p)
    assert abs(ynew[0] - y(tn + dt)) < 1e-13 * max(1, abs(y(tn + dt)))
    assert abs(e[0]) < 1e-13 * max(1, abs(y(tn + dt)))


def test_abm_error_constants_match_printed_values():
    """t^5: exact - p = (161/480) 5! dt^5, exact - c = -(9/480) 5! dt^5 (Eq. 78a, 78c);
    the modifier (161/170) and the final combination (9/170) cancel them (Eq. 78b, 78d)."""
    dt, tn = 0.5, 0.7
    y, f, arr = _poly_history(5, dt, tn)
    ep = GOLD["abm_predictor_error"]; ec = GOLD["abm_corrector_error"]
    e_n = arr(-(ep["num"] / ep["den"] - ec["num"] / ec["den"]) * 120 * dt ** 5)   # p_n - c_n for t^5
    p, m = ref.abm_predict(dt, arr(y(tn)), arr(y(tn - dt)), arr(f(tn)), arr(f(tn - dt)), arr(f(tn - 2 * dt)),
                           arr(f(tn - 3 * dt)), e_n)
    assert abs((y(tn + dt) - p[0]) / dt ** 5 - ep["num"] / ep["den"] * 120) < 1e-10
    assert abs(m[0] - y(tn + dt)) < 1e-12
    ynew, e = ref.abm_correct(dt, arr(y(tn)), arr(y(tn - dt)), arr(f(tn + dt)), arr(f(tn)), arr(f(tn - dt)),
                              arr(f(tn - 2 * dt)), p)
    c = p[0] - e[0]
    assert abs((y(tn + dt) - c) / dt ** 5 - ec["num"] / ec["den"] * 120) < 1e-10
    assert abs(ynew[0] - y(tn + dt)) < 1e-12
    assert abs(GOLD["abm_modifier_factor"]["num"] / GOLD["abm_modifier_factor"]["den"] - 161 / 170) == 0


def test_abm_linear_oscillator_phase_error():
    """y' = i w y with exact history: |y_n - e^{i w t_n}| <= ~ n 0.0098 |w dt|^6, stable."""
    w, dt = 1.0, 0.1
    arr = lambda v: np.array([v], dtype=complex)
    ex = lambda t: np.exp(1j * w * t)
    fx = lambda t: 1j * w * ex(t)
    yn, ym1 = arr(ex(0)), arr(ex(-dt))
    fh = [arr(fx(-dt)), arr(fx(-2 * dt)), arr(fx(-3 * dt))]
    e = arr(0.0)
    n = 200
    for s in range(n):
        f_n = 1j * w * yn
        p, m = ref.abm_predict(dt, yn, ym1, f_n, fh[0], fh[1], fh[2], e)
        ynew, e = ref.abm_correct(dt, yn, ym1, 1j * w * m, f_n, fh[0], fh[1], p)
        ym1, yn = yn, ynew
        fh = [f_n, fh[0], fh[1]]
    err = abs(yn[0] - ex(n * dt))
    assert err < 3 * n * 0.0098 * (w * dt) ** 6
    assert err > 0.05 * n * 0.0098 * (w * dt) ** 6     # and it is not better than the method allows
    # weak damping of the principal root: |mu| - 1 ~ -0.009 |z|^6 per step
    assert 0.006 < (1 - abs(yn[0])) / (n * (w * dt) ** 6) < 0.012


# ---------------------------------------------------------------------------------------------
# full stepper: free particles, invariants, time reversal
# ---------------------------------------------------------------------------------------------
def _free_params():
    par = ref.default_params()
    for k in ("t0", "t1", "t2", "t3", "W0", "g0_n", "g0_p"):
        setattr(par, k, 0.0)
    par.coulomb = 0
    return par


def test_free_two_mode_state_exact_phase():
    """interaction off: u_up = a e^{ik1.r}, v_up = b e^{ik2.r} evolve with e^{-i(E1-eta)t}, e^{+i(E2+eta)t},
    eta = |a|^2 V E1 - |b|^2 V E2 (Eqs. 11, 80, 81; run mode -i 2 of L1020)."""
    shape, a, dt = (8, 6, 4), 1.25, 0.05
    par = _free_params()
    c = ref.RefContext(*shape, a, dt, 1, 0, params=par)
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    Ls = [n * a for n in shape]
    k1 = np.array([2 * np.pi * 2 / Ls[0], 2 * np.pi * -1 / Ls[1], 0.0])
    k2 = np.array([2 * np.pi * -3 / Ls[0], 2 * np.pi * 2 / Ls[1], 2 * np.pi * 1 / Ls[2]])
    V = np.prod(Ls)
    A, B = 0.8 / math.sqrt(V), 0.6 / math.sqrt(V)
    pw = lambda q: np.exp(1j * sum(qi * xi for qi, xi in zip(q, x)))
    psi = np.zeros((1, 4) + shape, complex)
    psi[0, 0] = A * pw(k1); psi[0, 2] = B * pw(k2)
    c.set_wavefunctions(0, psi)
    E1, E2 = par.hbar2_2m * k1 @ k1, par.hbar2_2m * k2 @ k2
    eta = 0.64 * E1 - 0.36 * E2
    nsteps = 10
    c.step(nsteps)
    t = nsteps * dt
    got = c.get_wavefunctions(0)
    want = np.zeros_like(psi)
    want[0, 0] = psi[0, 0] * np.exp(-1j * (E1 - eta) * t / par.hbarc)
    want[0, 2] = psi[0, 2] * np.exp(+1j * (E2 + eta) * t / par.hbarc)
    z = max(abs(E1 - eta), abs(E2 + eta)) * dt / par.hbarc
    bound = 3 * z ** 5 / 120 + nsteps * 0.0098 * z ** 6
    err = np.abs(got - want).max() / np.abs(want).max()
    assert err < 5 * bound + 1e-13, (err, bound, z)
    # without phase removal the bare phases e^{-iE1 t}, e^{+iE2 t}
    par.remove_phase = 0
    c2 = ref.RefContext(*shape, a, dt, 1, 0, params=par)
    c2.set_wavefunctions(0, psi); c2.step(4)
    got2 = c2.get_wavefunctions(0)
    w2 = psi[0, 0] * np.exp(-1j * E1 * 4 * dt / par.hbarc)
    assert np.abs(got2[0, 0] - w2).max() / np.abs(w2).max() < 1e-8


def _defective_set(shape, dx, nwf, theta, scale):
    """an orthonormal set with two planted defects: state 3 <- cos(theta) psi_3 + sin(theta) e^{0.7 i} psi_4 (overlap
    <psi_3|psi_4> = sin(theta) e^{-0.7 i}, norm still 1) and state 1 <- scale psi_1 (norm scale^2, still orthogonal)."""
    from paper_2009_00745_b200 import inputs
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = shape; cfg["dx"] = dx
    psi = inputs.make_species(cfg, 0, nwf, seed=5).numpy().copy()
    psi[3] = math.cos(theta) * psi[3] + math.sin(theta) * np.exp(0.7j) * psi[4]
    psi[1] *= scale
    return psi


def test_norm_and_orthonormality_defects_have_their_closed_form_values():
    """lise_observables' defects: max_k |<psi_k|psi_k> - 1| and the largest sampled |<psi_k|psi_l>|
    (neighbours k + 1, k + 2 and k + nwf / 2) on a set with a planted overlap sin(theta) and a planted norm scale^2."""
    shape, dx, nwf, theta, scale = (8, 8, 8), 1.5, 6, 0.3, 1.05
    psi = _defective_set(shape, dx, nwf, theta, scale)
    c = ref.RefContext(*shape, dx, 0.05, nwf, 0)
    c.set_wavefunctions(0, psi)
    o = c.observables()
    assert abs(o["norm_defect"] - (scale ** 2 - 1.0)) < 1e-12
    assert abs(o["ortho_defect"] - math.sin(theta)) < 1e-12


def test_static_scf_solution_is_stationary():
    """SURVEY 8(c) "stationarity of a tiny static solution": a self-consistent Hartree-Fock state (pairing off,
    Coulomb on, 2 neutrons + 2 protons on 6^3) is built HERE by dense diagonalisation of the single-particle h of
    Eq. 12 (tests/dense_ref.py, Kronecker products of the closed-form Eq. 48 matrices) in the oracle's mean field,
    iterated with linear density mixing.  With v_k = conj(phi_k) of the occupied orbitals (Eq. 11: the v sector
    carries -h*) the oracle's time evolution must leave wavefunctions, densities and energy unchanged (Eqs. 80-81
    remove the phase e^{+i eps t}): this ties densities -> mean field -> H psi -> stepper into one loop."""
    from tests import dense_ref
    shape, a = (6, 6, 6), 1.6
    par = ref.default_params(); par.g0_n = 0.0; par.g0_p = 0.0
    c = ref.RefContext(*shape, a, 0.05, 2, 2, params=par)
    psi, eps, it, change = dense_ref.scf_ground_state(c, shape, a)
    assert change < 1e-13, (it, change)
    assert eps[0][1] < 0.0 and eps[1][1] < 0.0                     # bound orbitals (a Kramers pair each)
    assert abs(eps[0][0] - eps[0][1]) < 1e-8 and eps[1][0] > eps[0][0]   # Coulomb lifts the proton level
    for q in (0, 1):
        c.set_wavefunctions(q, psi[q])
    o0 = c.observables(); d0 = [c.densities(q) for q in (0, 1)]
    # H psi_k = -eps_k psi_k for the v-type states, to the accuracy of the self-consistency
    for q in (0, 1):
        hp = c.apply_h(q, psi[q]).reshape(psi[q].shape)
        for k in range(2):
            assert np.abs(hp[k] + eps[q][k] * psi[q][k]).max() < 1e-9 * abs(eps[q][k]) * np.abs(psi[q][k]).max() + 1e-11
    c.step(8)                                                    # 3 starter + 5 ABM steps
    for q in (0, 1):
        got = c.get_wavefunctions(q)
        assert np.abs(got - psi[q]).max() < 1e-11 * np.abs(psi[q]).max()          # measured 2e-14
        d1 = c.densities(q)
        assert np.abs(d1[0] - d0[q][0]).max() < 1e-12 * np.abs(d0[q][0]).max()
    o1 = c.observables()
    assert abs(o1["energy"] - o0["energy"]) < 1e-12 * abs(o0["energy"])
    # without phase removal the same state rotates with e^{+i eps t / hbar c} (v sector of Eq. 11)
    par.remove_phase = 0
    c2 = ref.RefContext(*shape, a, 0.05, 2, 2, params=par)
    for q in (0, 1):
        c2.set_wavefunctions(q, psi[q])
    c2.step(4)
    t = 4 * 0.05
    got = c2.get_wavefunctions(0)
    want = psi[0][0] * np.exp(1j * eps[0][0] * t / par.hbarc)
    assert np.abs(got[0] - want).max() < 1e-10 * np.abs(want).max()


def test_stepper_is_the_scalar_linear_recurrence_of_eq78_to_roundoff():
    """SURVEY 8(c) "ABM linear recurrence": interaction and phase removal off, one plane-wave state: H psi = E psi
    with a constant E, so the whole stepper (3 starter steps = multiplication by the 4th-order series T4(z), Eq. 77,
    then Eqs. 78a-d with its history rotation and e_3 = 0, reading B18) is a linear recurrence in one complex
    amplitude.  The recurrence is run here in scalar Python arithmetic and must agree to round-off, not to the
    truncation error: a swapped history slot, a stale e_n or a wrong hand-off from the starter fails at 1e-9."""
    shape, a, dt = (6, 4, 8), 1.25, 0.05
    par = _free_params()
    par.remove_phase = 0
    c = ref.RefContext(*shape, a, dt, 1, 0, params=par)
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    Ls = [n * a for n in shape]
    k = np.array([2 * np.pi * 2 / Ls[0], 2 * np.pi * 1 / Ls[1], 2 * np.pi * -3 / Ls[2]])
    psi = np.zeros((1, 4) + shape, complex)
    psi[0, 1] = np.exp(1j * sum(qi * xi for qi, xi in zip(k, x))) / math.sqrt(np.prod(Ls))
    c.set_wavefunctions(0, psi)
    lam = -1j * par.hbar2_2m * (k @ k) / par.hbarc           # y' = lam y  (Eq. 80 with eta = 0, u component)
    z = lam * dt
    T4 = 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24
    ys = [1.0 + 0j]
    for _ in range(3):
        ys.append(T4 * ys[-1])
    fs = [lam * y for y in ys]                               # f_0 .. f_3
    e = 0.0
    nabm = 9
    for n in range(3, 3 + nabm):
        pn = (ys[n] + ys[n - 1]) / 2 + dt / 48 * (119 * fs[n] - 99 * fs[n - 1] + 69 * fs[n - 2] - 17 * fs[n - 3])
        mn = pn - 161 / 170 * e
        cn = (ys[n] + ys[n - 1]) / 2 + dt / 48 * (17 * lam * mn + 51 * fs[n] + 3 * fs[n - 1] + fs[n - 2])
        e = pn - cn
        ys.append(cn + 9 / 170 * e)
        fs.append(lam * ys[-1])
    c.step(3 + nabm)
    got = c.get_wavefunctions(0)
    want = psi[0, 1] * ys[-1]
    assert np.abs(got[0, 1] - want).max() / np.abs(want).max() < 2e-13
    assert np.abs(got[0, [0, 2, 3]]).max() < 1e-15
    # and the recurrence itself tracks e^{lam t} within the method's error (so the pin is not vacuous)
    t = (3 + nabm) * dt
    assert abs(ys[-1] - np.exp(lam * t)) < 5 * (3 * abs(z) ** 5 / 120 + nabm * 0.0098 * abs(z) ** 6)


@pytest.fixture(scope="module")
def evolved_small():
    """config-0-like small problem: both species, Coulomb, pairing, 10 steps."""
    from paper_2009_00745_b200 import inputs
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (8, 8, 10); cfg["dx"] = 1.5
    psi = [inputs.make_species(cfg, q, 12, seed=99).numpy() for q in (0, 1)]
    c = ref.RefContext(*cfg["shape"], cfg["dx"], 0.05, 12, 12)
    for q in (0, 1):
        c.set_wavefunctions(q, psi[q])
    o0 = c.observables()
    c.step(10)
    o1 = c.observables()
    return c, psi, o0, o1


def test_norm_and_orthonormality_preserved(evolved_small):
    """one Hermitian H for all states and real eta_k: norms and overlaps conserved to truncation."""
    c, psi, o0, o1 = evolved_small
    assert o0["norm_defect"] < 1e-13 and o0["ortho_defect"] < 1e-13
    assert o1["norm_defect"] < 1e-11 and o1["ortho_defect"] < 1e-11
    assert o1["step"] == 10 and abs(o1["time"] - 0.5) < 1e-15


def test_energy_and_number_drift_small_for_incomplete_set(evolved_small):
    """random incomplete sets with pairing drift slightly in the exact equations (SURVEY finding 8);
    the drift stays far below the scale of the energy."""
    c, psi, o0, o1 = evolved_small
    assert abs(o1["energy"] - o0["energy"]) < 1e-4 * abs(o0["energy"])
    assert abs(o1["n_neutron"] - o0["n_neutron"]) < 1e-4 * o0["n_neutron"]
    assert abs(o1["n_proton"] - o0["n_proton"]) < 1e-4 * o0["n_proton"]


def test_energy_number_conserved_pairing_off_and_time_reversal():
    """pairing off: E and N conserved to truncation for any set; forward then backward in time
    recovers the initial wavefunctions and energy (L663)."""
    from paper_2009_00745_b200 import inputs
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (8, 8, 8); cfg["dx"] = 1.5
    psi = [inputs.make_species(cfg, q, 8, seed=5).numpy() for q in (0, 1)]
    par = ref.default_params(); par.g0_n = 0.0; par.g0_p = 0.0
    c = ref.RefContext(*cfg["shape"], cfg["dx"], 0.04, 8, 8, params=par)
    for q in (0, 1):
        c.set_wavefunctions(q, psi[q])
    o0 = c.observables()
    c.step(8)
    o1 = c.observables()
    assert abs(o1["energy"] - o0["energy"]) < 1e-9 * abs(o0["energy"])
    assert abs(o1["n_neutron"] - o0["n_neutron"]) < 1e-11 * o0["n_neutron"]
    c.set_dt(-0.04)
    c.step(8)
    o2 = c.observables()
    assert abs(o2["energy"] - o0["energy"]) < 1e-9 * abs(o0["energy"])
    back = c.get_wavefunctions(0)
    # states return up to the (state-dependent, removed) global phase: compare overlaps
    ov = np.abs(np.einsum("kcxyz,kcxyz->k", np.conj(back), psi[0])) * cfg["dx"] ** 3
    assert np.abs(ov - 1).max() < 1e-7


def test_starter_is_third_order():
    """starter only (3 series-expansion steps with the midpoint Hamiltonian, Eqs. 75-77, reading B18): the error after
    the 3 steps against a fine reference at the same final time is O(dt^3); halving dt divides it by 8-9 (SURVEY 8(c)
    states an observed ratio of about 9)."""
    from paper_2009_00745_b200 import inputs
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (6, 6, 6); cfg["dx"] = 1.5
    psi = inputs.make_species(cfg, 0, 6, seed=3).numpy()

    def run(dt, n):
        c = ref.RefContext(*cfg["shape"], cfg["dx"], dt, 6, 0)
        c.set_wavefunctions(0, psi); c.step(n)
        w = c.get_wavefunctions(0); c.close()
        return w

    def starter_error(dt):
        return np.abs(run(dt, 3) - run(3 * dt / 48, 48)).max()

    e1, e2 = starter_error(0.2), starter_error(0.1)
    assert 7.0 < e1 / e2 < 10.0, (e1, e2, e1 / e2)
