"""Pins of the oracle's "next" features against closed forms and identities (CPU only, no CUDA):
restart / renormalisation / observables of Eqs. 37-41, functional variants of Eqs. 8, 10, 15, 20
(8(f)3), boosts, external fields, moving and rotating frames of Eqs. 23-36 (8(f)4).
"""
import cmath
import math

import numpy as np
import pytest
import scipy.integrate

from oracle import ref
from tests.test_oracle_pins import _free_params, _smooth_states


def _gauss(shape, a, centre, sig):
    x = [np.arange(n) * a for n in shape]                              # Eq. 43: x_i = i a
    g = [np.exp(-(x[i] - centre[i]) ** 2 / (2 * sig[i] ** 2)) / (math.sqrt(2 * math.pi) * sig[i]) for i in range(3)]
    return g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :]


# ---------------------------------------------------------------------------------------------
# (f)2: observables of Eqs. 37-41
# ---------------------------------------------------------------------------------------------
def test_moments_of_displaced_gaussians_closed_form():
    """Eqs. 37, 38b-e, 39, 40, 27, 41 on Gaussian densities (lattice sums of well-resolved Gaussians are exact to
    round-off): a wrong origin, a missing r - R_cm shift, a swapped Q_lm polynomial or a wrong hbar / m factor fails."""
    shape, a = (24, 24, 28), 1.0
    c = ref.RefContext(*shape, a, 0.05, 1, 1)
    cn, cp, sg = (11.3, 12.1, 13.7), (11.9, 11.5, 14.6), (1.35, 1.4, 1.45)
    Nn, Np = 7.0, 5.0
    q = np.array([0.11, -0.07, 0.19])                                   # uniform flow: j = q n
    dn, dp = np.zeros((14,) + shape), np.zeros((14,) + shape)
    dn[0], dp[0] = Nn * _gauss(shape, a, cn, sg), Np * _gauss(shape, a, cp, sg)
    for i in range(3):
        dn[6 + i], dp[6 + i] = q[i] * dn[0], q[i] * dp[0]
    pn, pp = np.zeros((14,) + shape), np.zeros((14,) + shape)
    pn[12], pn[13] = 0.6, -0.8                                          # |Delta_n| = 1.0
    pp[12] = 0.5                                                        # |Delta_p| = 0.5
    o = c.moments_from(dn, dp, pn, pp)
    A = Nn + Np
    rcm = (Nn * np.array(cn) + Np * np.array(cp)) / A
    assert np.abs(np.array(o["rcm_n"]) - cn).max() < 1e-11 and np.abs(np.array(o["rcm_p"]) - cp).max() < 1e-11
    assert np.abs(np.array(o["rcm"]) - rcm).max() < 1e-11
    assert abs(o["delta_n"] - 1.0) < 1e-13 and abs(o["delta_p"] - 0.5) < 1e-13
    h2m, hbarc = c.params.hbar2_2m, c.params.hbarc
    assert abs(o["e_coll"] - h2m * q @ q * A) < 1e-11 * h2m * A         # Eq. 40: (hbar^2/2m) j^2 / n = (hbar^2 q^2/2m) n
    assert np.abs(np.array(o["v_cm"]) - 2 * h2m / hbarc * q).max() < 1e-14   # Eq. 27: hbar q / m in units of c
    assert abs(o["e_cm"] - h2m * q @ q * A) < 1e-11 * h2m * A           # Eq. 41: a rigid flow has E_cm = E_coll
    # multipoles of the two-Gaussian mixture about the total centre of mass, from the Gaussian moments
    var = np.array(sg) ** 2

    def mom(cen, N):
        d = np.array(cen) - rcm
        m2 = var + d * d                                                # <x_i^2>
        m4 = 3 * var ** 2 + 6 * var * d * d + d ** 4                    # <x_i^4>
        m3z = d[2] ** 3 + 3 * d[2] * var[2]
        q20 = 2 * m2[2] - m2[0] - m2[1]
        q30 = 2 * m3z - 3 * d[2] * (m2[0] + m2[1])
        zz_r2 = m4[2] + m2[2] * (m2[0] + m2[1])
        r4 = m4.sum() + 2 * (m2[0] * m2[1] + m2[0] * m2[2] + m2[1] * m2[2])
        q40 = 35 * m4[2] - 30 * zz_r2 + 3 * r4
        return N * np.array([q20, q30, q40, d[0] * d[2], d[1] * d[2], m2[0] - m2[1], 2 * d[0] * d[1]])
    want = mom(cn, Nn) + mom(cp, Np)
    got = np.array([o["q20"], o["q30"], o["q40"], o["q21"][0], o["q21"][1], o["q22"][0], o["q22"][1]])
    assert np.abs(got - want).max() < 1e-10 * np.abs(want).max()
    c.close()


def test_restart_goes_through_the_starter_and_keeps_the_clock():
    """L764-L768: a restart saves only the latest wavefunctions and re-enters through the series expansion; the
    restarted run equals a fresh run from y_k bit for bit, keeps time and step count, and stays on the trajectory of
    the uninterrupted run to the starter's O(dt^3)."""
    from paper_2009_00745_b200 import inputs
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (6, 6, 8)
    psi = inputs.make_species(cfg, 0, 5, seed=4).numpy()
    dt = 0.05
    a = ref.RefContext(*cfg["shape"], cfg["dx"], dt, 5, 0)
    a.set_wavefunctions(0, psi); a.step(5)
    y5 = a.get_wavefunctions(0)
    a.step(3)
    y8_uninterrupted = a.get_wavefunctions(0)
    b = ref.RefContext(*cfg["shape"], cfg["dx"], dt, 5, 0)
    b.set_wavefunctions(0, y5); b.set_time(5 * dt, 5); b.step(3)
    fresh = ref.RefContext(*cfg["shape"], cfg["dx"], dt, 5, 0)
    fresh.set_wavefunctions(0, y5); fresh.step(3)
    assert np.array_equal(b.get_wavefunctions(0), fresh.get_wavefunctions(0))
    ob = b.observables()
    assert ob["step"] == 8 and abs(ob["time"] - 8 * dt) < 1e-15
    dev = np.abs(b.get_wavefunctions(0) - y8_uninterrupted).max() / np.abs(y8_uninterrupted).max()
    assert 0.0 < dev < 1e-5
    for ctx in (a, b, fresh):
        ctx.close()


def test_renormalisation_is_a_rescaling_at_the_end_of_the_step():
    """L637: with renormalize on, y_{n+1} is the plain step's y_{n+1} divided by its norm, state by state."""
    from paper_2009_00745_b200 import inputs
    cfg = dict(inputs.CONFIGS[0]); cfg["shape"] = (6, 6, 6)
    psi = 1.001 * inputs.make_species(cfg, 0, 4, seed=9).numpy()       # slightly off-norm input
    plain = ref.RefContext(*cfg["shape"], cfg["dx"], 0.05, 4, 0)
    plain.set_wavefunctions(0, psi); plain.step(1)
    y = plain.get_wavefunctions(0)
    par = ref.default_params(); par.coulomb = 0; par.renormalize = 1
    rn = ref.RefContext(*cfg["shape"], cfg["dx"], 0.05, 4, 0, params=par)
    rn.set_wavefunctions(0, psi); rn.step(1)
    nrm = np.sqrt((np.abs(y) ** 2).sum(axis=(1, 2, 3, 4), keepdims=True) * cfg["dx"] ** 3)
    assert np.abs(rn.get_wavefunctions(0) - y / nrm).max() < 1e-15
    rn.step(4)
    assert rn.observables()["norm_defect"] < 5e-15
    plain.close(); rn.close()


# ---------------------------------------------------------------------------------------------
# (f)3: functional variants
# ---------------------------------------------------------------------------------------------
def test_spherical_cutoff_geff_equals_the_regulated_integral():
    """Eq. 20a for k_F^2 >= 0: 1/g_eff = 1/g0 - int_{k<k_c} d^3k/(2 pi)^3 1 / (2 (eps_k - mu)) (principal value) with
    eps_k = hbar^2 k^2 / 2 m* + U; for k_F^2 < 0 the printed arctan form is the analytic continuation k_F -> i |k_F|."""
    g0, M, U = -250.0, 18.5, -40.0
    for mu, ec in ((-8.0, 60.0), (-39.0, 25.0), (5.0, 80.0)):
        kf, kc = math.sqrt((mu - U) / M), math.sqrt((ec + mu - U) / M)
        pv, _ = scipy.integrate.quad(lambda k: 1.0 / (k + kf), 0.0, kc, weight="cauchy", wvar=kf, epsabs=1e-13)
        integral = (kc + kf * kf * pv) / (4 * math.pi ** 2 * M)      # (4 pi / (2 pi)^3) int k^2 dk / (2 M (k^2 - kF^2))
        assert abs(ref.inv_geff_spherical(g0, M, U, mu, ec) - (1 / g0 - integral)) < 1e-12
    for mu, ec in ((-55.0, 70.0), (-41.0, 30.0)):
        kc, kap = math.sqrt((ec + mu - U) / M), math.sqrt((U - mu) / M)
        kfc = 1j * kap
        br = 1 - kfc / (2 * kc) * cmath.log((kc + kfc) / (kc - kfc))
        assert abs(br.imag) < 1e-15
        assert abs(ref.inv_geff_spherical(g0, M, U, mu, ec) - (1 / g0 - kc / (4 * math.pi ** 2 * M) * br.real)) < 1e-15
    # continuity across k_F = 0 and no pairing above the cutoff
    lo, hi = ref.inv_geff_spherical(g0, M, U, U - 1e-9, 50.0), ref.inv_geff_spherical(g0, M, U, U + 1e-9, 50.0)
    assert abs(lo - hi) < 1e-8
    assert ref.inv_geff_spherical(g0, M, 100.0, -8.0, 60.0) == 0.0


def test_lattice_cutoff_geff_counter_term_is_the_momentum_integral_over_the_brillouin_cube():
    """Eq. 21, pinned without K and without retyping its prefactor: the term subtracted from 1/g0 is
    the free-particle pairing loop regulated by the lattice's own momentum cutoff, every |k_i| <= pi/a:
        1/g0 - 1/g_eff = int_{|k_i| <= pi/a} d^3k / (2 pi)^3  1 / (2 M k^2),    M = hbar^2 / 2 m*(r)
    (the same integral that Eq. 20 cuts off spherically).  With k = (pi/a) x this is I / (16 pi^2 a M) with
    I = int_{[-1,1]^3} d^3x / |x|^2.  Radially, int_0^R dr r^2 / r^2 = R(direction), and over the pyramid under the face
    z = 1, with (u, v, 1) the point where the ray leaves the cube, dOmega = du dv / (1+u^2+v^2)^(3/2) and R = sqrt(1+u^2+v^2):
        I = 6 int_{-1}^{1} int_{-1}^{1} du dv / (1 + u^2 + v^2)    -- a smooth 2-D quadrature, done here.
    The oracle side is read off its outputs: Delta = -g_eff kappa (Eq. 19), so 1/g0 - 1/g_eff = 1/g0 + kappa/Delta.  A wrong
    factor in the m* <-> M conversion, in the powers of pi or in a fails this."""
    import scipy.integrate
    I2, err = scipy.integrate.dblquad(lambda v, u: 1.0 / (1.0 + u * u + v * v), -1.0, 1.0, -1.0, 1.0, epsabs=1e-13, epsrel=1e-13)
    I = 6.0 * I2
    # coarse brute-force guard of the reduction itself: midpoint rule of 1/|x|^2 on the cube (the singularity is integrable;
    # the rule converges like h), compared at 1e-2
    n = 96
    x = (np.arange(n) + 0.5) / n
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    brute = 8.0 * (1.0 / (X * X + Y * Y + Z * Z)).sum() / n ** 3
    assert abs(brute - I) < 1e-2 * I, (brute, I)
    shape, a = (10, 10, 12), 1.25
    rng = np.random.default_rng(21)
    for a in (1.25, 1.0):
        par = ref.default_params(); par.coulomb = 0                    # alpha_pair = 0: g0(r) = g0 (Eq. 8)
        c = ref.RefContext(*shape, a, 0.05, 1, 1, params=par)
        dn, dp = _smooth_densities(shape, a, rng)
        pots = c.potentials_from(dn, dp)
        for q, d, g0 in ((0, dn, par.g0_n), (1, dp, par.g0_p)):
            M = pots[q][1]
            assert M.max() - M.min() > 0.5                             # m*(r) really varies over the box
            kappa = d[12] + 1j * d[13]
            delta = pots[q][12] + 1j * pots[q][13]
            counter = 1.0 / g0 + kappa / delta
            want = I / (16.0 * math.pi ** 2 * a * M)
            assert np.abs(counter.imag).max() < 1e-12 * np.abs(want).max()
            assert np.abs(counter.real - want).max() < 1e-8 * np.abs(want).max(), (q, a)
        c.close()


def _fd_du(c, dn, dp, q, delta, eps=1e-5):
    """(E[n_q + eps delta] - E[n_q - eps delta]) / 2 eps at fixed other fields, and dV sum U_q delta."""
    d = [dn, dp]
    e = []
    for sgn in (+1, -1):
        x = [a.copy() for a in d]
        x[q][0] += sgn * eps * delta
        e.append(c.potentials_from(x[0], x[1])[2][0])
    pots = c.potentials_from(dn, dp)
    return (e[0] - e[1]) / (2 * eps), (pots[q][0] * delta).sum() * c.dx ** 3


def _smooth_densities(shape, a, rng):
    dn, dp = np.zeros((14,) + shape), np.zeros((14,) + shape)
    base = _gauss(shape, a, [0.5 * n * a for n in shape], (2.2, 2.5, 2.0))
    dn[0] = 9.0 * base + 1e-3
    dp[0] = 6.0 * _gauss(shape, a, [0.5 * n * a + 0.4 for n in shape], (2.0, 2.3, 2.1)) + 1e-3
    for d in (dn, dp):
        d[12] = 0.02 * base * rng.uniform(0.5, 1.0)                       # kappa (re, im)
        d[13] = 0.015 * base * rng.uniform(0.5, 1.0)
    return dn, dp


def test_seall1_mean_field_is_the_derivative_of_its_energy():
    """Eq. 15 (as printed) = d E_vol / d n_q of Eq. 10 with (n1/n0)^(2j) (reading B29), plus the gradient term."""
    shape, a = (10, 10, 12), 1.25
    rng = np.random.default_rng(5)
    par = ref.default_params()
    par.functional = 1; par.coulomb = 0; par.g0_n = par.g0_p = 0.0
    par.sea_a[:] = (-420.0, 190.0, -60.0); par.sea_b[:] = (-310.0, 220.0, 80.0); par.sea_c[:] = (610.0, -140.0, 35.0)
    par.sea_cdn[:] = (-55.0, 12.0); par.sea_cdj[:] = (-70.0, -25.0)
    c = ref.RefContext(*shape, a, 0.05, 1, 1, params=par)
    dn, dp = _smooth_densities(shape, a, rng)
    for q in (0, 1):
        delta = _gauss(shape, a, (5.0, 6.0, 7.0), (1.8, 1.6, 2.0))
        fd, an = _fd_du(c, dn, dp, q, delta)
        assert abs(fd - an) < 1e-7 * abs(an), (q, fd, an)
    # m* = m for SeaLL1 (L135): the kinetic field is the bare hbar^2 / 2m
    assert np.abs(c.potentials_from(dn, dp)[0][1] - par.hbar2_2m).max() == 0.0
    c.close()


@pytest.mark.parametrize("alpha", [0.5, 1.0])
def test_density_dependent_pairing_coupling_enters_the_mean_field(alpha):
    """Eq. 8 with alpha != 0: U = dE/dn_q must contain |kappa|^2 d g_eff / d n through g0(n) (and through m*)."""
    shape, a = (10, 10, 12), 1.25
    rng = np.random.default_rng(6)
    par = ref.default_params(); par.coulomb = 0; par.alpha_pair = alpha
    c = ref.RefContext(*shape, a, 0.05, 1, 1, params=par)
    dn, dp = _smooth_densities(shape, a, rng)
    pots = c.potentials_from(dn, dp)
    g0r = par.g0_n * (1 - alpha * (dn[0] + dp[0]) / 0.16)
    geff = 1 / (1 / g0r - ref.pairing_K() / (8 * math.pi * a * pots[0][1]))
    assert np.abs(pots[0][12] + geff * dn[12]).max() < 1e-13 * np.abs(pots[0][12]).max()   # Eq. 19 with Eq. 8 in Eq. 21
    for q in (0, 1):
        delta = _gauss(shape, a, (6.0, 6.0, 7.0), (1.8, 1.6, 2.0))
        fd, an = _fd_du(c, dn, dp, q, delta)
        assert abs(fd - an) < 1e-7 * abs(an), (q, fd, an)
    c.close()


# ---------------------------------------------------------------------------------------------
# (f)4: boosts, external fields, frames
# ---------------------------------------------------------------------------------------------
def test_boost_is_the_gauge_transformation_of_eq_23():
    """Eq. 23 with chi = q.r: n unchanged, j -> j + q n, and the collective energy of Eq. 40 rises by (hbar^2 q^2/2m) N
    for a state at rest."""
    shape, a = (8, 8, 10), 1.25
    rng = np.random.default_rng(7)
    psi = _smooth_states(shape, a, 3, rng, kc=1.2)
    psi = np.concatenate([psi[:, :2].real, psi[:, 2:].real], axis=1).astype(complex)   # real states: j = 0
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2, 3, 4), keepdims=True) * a ** 3)
    c = ref.RefContext(*shape, a, 0.05, 3, 0, params=_free_params())
    c.set_wavefunctions(0, psi)
    d0 = c.densities(0)
    m = (1, 0, -1)
    q = np.array([2 * np.pi * m[i] / (shape[i] * a) for i in range(3)])
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    chi = sum(q[i] * x[i] for i in range(3))
    c.boost(0, chi)
    want = psi.copy(); want[:, :2] *= np.exp(1j * chi); want[:, 2:] *= np.exp(-1j * chi)
    assert np.abs(c.get_wavefunctions(0) - want).max() < 1e-15
    d1 = c.densities(0)
    assert np.abs(d1[0] - d0[0]).max() < 1e-14 and np.abs(d0[6:9]).max() < 1e-14
    for i in range(3):
        assert np.abs(d1[6 + i] - q[i] * d0[0]).max() < 1e-13
    o = c.observables_ext()
    N = d0[0].sum() * a ** 3
    assert abs(o["e_coll"] - c.params.hbar2_2m * q @ q * N) < 1e-11
    c.close()


def test_frame_terms_closed_forms_on_free_states():
    """Eqs. 24, 26, 36 with the interaction off: (i) -v.p shifts a plane wave's energy by -hbar c v.k; (ii) -omega.s
    is -(hbar c / 2) omega.sigma; (iii) -omega.l acts on an l_z = 1 function about the origin as -hbar c omega_z;
    (iv) a scalar field adds U0 psi.  Signs and the factor of A = -(hbar c / 2) Uvec are what these pin."""
    shape, a = (16, 16, 8), 0.9
    par = _free_params()
    c = ref.RefContext(*shape, a, 0.05, 1, 0, params=par)
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    hbarc, h2m = par.hbarc, par.hbar2_2m
    # (i) + (iv)
    k = np.array([2 * np.pi * 2 / (shape[0] * a), -2 * np.pi * 1 / (shape[1] * a), 2 * np.pi * 1 / (shape[2] * a)])
    pw = np.exp(1j * sum(k[i] * x[i] for i in range(3)))
    psi = np.zeros((1, 4) + shape, complex); psi[0, 0] = pw
    v = np.array([0.02, -0.05, 0.03])
    u0 = 3.0 + np.cos(2 * np.pi * x[0] / (shape[0] * a))
    c.set_wavefunctions(0, psi)
    c.set_frame(v_cm=v)
    c.set_external_fields(0, u0=u0)
    h = c.apply_h(0, psi).reshape(psi.shape)
    assert np.abs(h[0, 0] - (h2m * k @ k - hbarc * v @ k + u0) * pw).max() < 1e-11
    # the same velocity given as a uniform external vector field (Eq. 24 with Uvec = v) is the same operator
    c.set_frame()
    c.set_external_fields(0, u0=u0, uvec=np.stack([np.full(shape, v[i]) for i in range(3)]))
    assert np.abs(c.apply_h(0, psi).reshape(psi.shape) - h).max() < 1e-12
    # the v components see -h^*: for the component v_up = conj(pw) the same plane wave phi = pw enters h
    psi2 = np.zeros((1, 4) + shape, complex); psi2[0, 2] = np.conj(pw)
    h2 = c.apply_h(0, psi2).reshape(psi.shape)
    assert np.abs(h2[0, 2] + np.conj((h2m * k @ k - hbarc * v @ k + u0) * pw)).max() < 1e-11
    # (ii)
    c.set_external_fields(0)
    om = np.array([0.0, 0.0, 0.004])
    c.set_frame(omega=om, origin=(0.0, 0.0, 0.0))
    const = np.zeros((1, 4) + shape, complex); const[0, 0] = 1.0
    # a constant has l = 0 on the lattice too: D (omega x r) . 1 + (omega x r) . D 1 = div(omega x r) = 0 row by row
    hc = c.apply_h(0, const).reshape(psi.shape)
    assert np.abs(hc[0, 0] + 0.5 * hbarc * om[2]).max() < 1e-11 and np.abs(hc[0, 1]).max() < 1e-11
    c.close()
    # (iii) f = ((x - x0) + i (y - y0)) exp(-r^2 / 2 s^2): l_z f = hbar f.  Lattice 32 x 32 with s chosen so that both the
    # Gaussian's tail at the box edge and its spectrum at the Nyquist mode are below 1e-10
    shape, a, sig = (32, 32, 4), 0.8, 1.75
    c = ref.RefContext(*shape, a, 0.05, 1, 0, params=par)
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    o = np.array([0.5 * shape[0] * a, 0.5 * shape[1] * a, 0.0])
    env = np.exp(-((x[0] - o[0]) ** 2 + (x[1] - o[1]) ** 2) / (2 * sig ** 2))
    f = ((x[0] - o[0]) + 1j * (x[1] - o[1])) * env
    st = np.zeros((1, 4) + shape, complex); st[0, 0] = f
    c.set_wavefunctions(0, st)
    c.set_frame(omega=om, origin=o)
    hf = c.apply_h(0, st).reshape(st.shape)
    c.set_frame()
    hf0 = c.apply_h(0, st).reshape(st.shape)
    assert np.abs((hf - hf0)[0, 0] - (-hbarc * om[2] - 0.5 * hbarc * om[2]) * f).max() < 1e-8 * np.abs(f).max() * hbarc * om[2]
    c.close()


def test_h_with_external_terms_is_hermitian_and_energy_of_external_terms():
    """with random external fields and frame terms H stays Hermitian, and e_ext = sum_k <phi_k| h_ext |phi_k>."""
    shape, a = (6, 8, 6), 1.25
    rng = np.random.default_rng(8)
    psi = _smooth_states(shape, a, 4, rng, kc=1.5)
    c = ref.RefContext(*shape, a, 0.05, 4, 0)
    c.set_wavefunctions(0, psi)
    u0 = rng.uniform(-5, 5, shape); uv = rng.uniform(-0.05, 0.05, (3,) + shape)
    c.set_external_fields(0, u0=u0, uvec=uv)
    c.set_frame(v_cm=(0.01, -0.02, 0.03), omega=(0.002, -0.001, 0.003), origin=(2.0, 3.0, 1.0))
    va = _smooth_states(shape, a, 1, rng, kc=3.0); vb = _smooth_states(shape, a, 1, rng, kc=3.0)
    ha, hb = c.apply_h(0, va), c.apply_h(0, vb)
    assert abs(np.vdot(va, hb) - np.conj(np.vdot(vb, ha))) < 1e-12 * abs(np.vdot(va, hb))
    h_with = c.apply_h(0, psi).reshape(psi.shape)
    pots_with = c.potentials(0)
    e_ext = c.observables_ext()["e_ext"]
    c.set_external_fields(0); c.set_frame()
    h_without = c.apply_h(0, psi).reshape(psi.shape)
    # H is the HFB matrix: the v block carries -h^*, so sum_k <phi_k|h_ext|phi_k> = - sum_k <v_k|(H_with - H_without) v_k>
    dh = h_with - h_without
    want = -np.real(np.vdot(psi[:, 2:], dh[:, 2:])) * a ** 3
    assert abs(e_ext - want) < 1e-10 * max(abs(want), 1.0)
    assert np.abs(pots_with[0] - c.potentials(0)[0] - u0).max() < 1e-12
    c.close()


def test_driven_free_state_follows_the_closed_form_phase_to_fourth_order():
    """PAPER.md:L232 (Eq. 24 with U(r, t)): a uniform field U0 f(t) on the free two-mode state u_up = A e^{ik1.r},
    v_up = B e^{ik2.r} (no phase removal) gives u(t) = u(0) exp(-i [E1 t + U0 F(t)] / hbar c) and
    v(t) = v(0) exp(+i [E2 t + U0 F(t)] / hbar c), F = int_0^t f.  With the amplitude pair (f(t_n), f(t_{n+1})) supplied
    before every step and an exact multistep history, the ABM error falls by >= 2^4 when dt is halved; with the starter
    it falls like the starter's own third order; a field frozen at t_n during the step is only first order."""
    shape, a = (8, 6, 4), 1.25
    par = _free_params(); par.remove_phase = 0
    x = np.meshgrid(*[np.arange(n) * a for n in shape], indexing="ij")
    Ls = [n * a for n in shape]
    k1 = np.array([2 * np.pi * 1 / Ls[0], 2 * np.pi * -1 / Ls[1], 0.0])
    k2 = np.array([2 * np.pi * -1 / Ls[0], 0.0, 2 * np.pi * 1 / Ls[2]])
    V = np.prod(Ls)
    pw = lambda q: np.exp(1j * sum(qi * xi for qi, xi in zip(q, x)))
    psi0 = np.zeros((1, 4) + shape, complex)
    psi0[0, 0] = 0.8 / math.sqrt(V) * pw(k1); psi0[0, 2] = 0.6 / math.sqrt(V) * pw(k2)
    E1, E2 = par.hbar2_2m * k1 @ k1, par.hbar2_2m * k2 @ k2
    U0, w = 40.0, 0.9                                   # MeV; f(t) = cos(w t) + 0.3 t, F(t) = sin(w t) / w + 0.15 t^2
    f = lambda t: math.cos(w * t) + 0.3 * t
    F = lambda t: math.sin(w * t) / w + 0.15 * t * t
    hc = par.hbarc

    def exact(t):
        y = np.zeros_like(psi0)
        y[0, 0] = psi0[0, 0] * np.exp(-1j * (E1 * t + U0 * F(t)) / hc)
        y[0, 2] = psi0[0, 2] * np.exp(+1j * (E2 * t + U0 * F(t)) / hc)
        return y

    def rhs(t):                                         # dy/dt of the exact solution
        y = exact(t); g = np.zeros_like(y)
        g[0, 0] = -1j * (E1 + U0 * f(t)) / hc * y[0, 0]
        g[0, 2] = +1j * (E2 + U0 * f(t)) / hc * y[0, 2]
        return g

    def run(dt, T, history, frozen=False):
        c = ref.RefContext(*shape, a, dt, 1, 0, params=par)
        c.set_external_fields(0, u0=np.full(shape, U0))
        c.set_wavefunctions(0, exact(0.0))
        n = int(round(T / dt))
        if history:                                     # exact y_{-1}, f_{-1..-3}, e_0 = 0: the ABM formulas alone
            c.set_history(0, exact(-dt), rhs(-dt), rhs(-2 * dt), rhs(-3 * dt), np.zeros_like(psi0))
        for i in range(n):
            t = i * dt
            c.set_external_amplitudes(f(t), f(t) if frozen else f(t + dt))
            c.step(1)
        got = c.get_wavefunctions(0)
        c.close()
        return np.abs(got - exact(n * dt)).max() / np.abs(psi0).max()

    T = 1.6
    e1, e2 = run(0.2, T, True), run(0.1, T, True)
    assert e2 < 2e-6 and e1 / e2 > 16.0, (e1, e2)                   # fourth order or better
    s1, s2 = run(0.2, T, False), run(0.1, T, False)
    assert 5.0 < s1 / s2 < 20.0 and s2 < 1e-4, (s1, s2)             # the starter's third order
    z1, z2 = run(0.2, T, True, frozen=True), run(0.1, T, True, frozen=True)
    assert 1.6 < z1 / z2 < 2.6 and z2 > 100 * e2, (z1, z2)          # what a per-step snapshot gives: first order
    # amplitudes (1, 1) are the static field of lise_ref_set_external_fields
    c = ref.RefContext(*shape, a, 0.05, 1, 0, params=par)
    c.set_external_fields(0, u0=np.full(shape, U0)); c.set_wavefunctions(0, psi0); c.step(4)
    want = psi0[0, 0] * np.exp(-1j * (E1 + U0) * 0.2 / hc)
    assert np.abs(c.get_wavefunctions(0)[0, 0] - want).max() / np.abs(want).max() < 1e-8
    c.close()
