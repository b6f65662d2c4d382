"""Seeded synthetic quasiparticle wavefunctions (the input recipe of DESIGN.md).

This module holds NONE of the method's arithmetic (no derivatives, densities, potentials, H or ABM):
it only draws counter-based random Fourier coefficients, multiplies by a Gaussian envelope and
orthonormalises.  It serves both the CPU oracle (tests) and the CUDA path (tests, bench), which is
the one thing the two are allowed to share.  torch is used for tensor plumbing on CPU or GPU.

Stand-in for the paper's real inputs (static SLDA solutions wf_*.cwr of 240Pu / 120Sn+120Sn,
PAPER.md L1070-L1083), which are not available.  Value distribution of the coefficients: uniform(-1,1)
real and imaginary parts, the paper's own noise distribution.
"""
import math

import torch

SEED0 = 20090745

# BASELINE.json configs with the deviations of SURVEY.md 8(d) (each reported in DESIGN.md)
CONFIGS = [
    dict(name="config0_12c_n128", shape=(12, 12, 12), dx=1.5, dt=0.05, steps=10, nwf=(128, 0),
         kc=0.8, w=4.0, centres=[(0.0, 0.0, 0.0)], occ=(0.5, 0.5), coulomb=False),
    dict(name="config1_24c", shape=(24, 24, 24), dx=1.25, dt=0.05, steps=100, nwf=(4096, 4096),
         kc=2.0, w=5.0, centres=[(0.0, 0.0, 0.0)], occ=None, coulomb=True, ortho="split"),
    dict(name="config2_32c", shape=(32, 32, 32), dx=1.25, dt=0.05, steps=100, nwf=(8192, 8192),
         kc=1.8, w=6.0, centres=[(0.0, 0.0, 0.0)], occ=None, coulomb=True, ortho="split"),
    dict(name="config3_24x24x64", shape=(24, 24, 64), dx=1.25, dt=0.05, steps=200, nwf=(8192, 8192),
         kc=1.2, w=4.0, centres=[(0.0, 0.0, -12.0), (0.0, 0.0, 12.0)], occ=None, coulomb=True, ortho="split"),
    dict(name="config4_40c", shape=(40, 40, 40), dx=1.0, dt=0.03, steps=100, nwf=(6144, 6144),
         kc=1.8, w=7.0, centres=[(0.0, 0.0, 0.0)], occ=None, coulomb=True, ortho="split"),
]
# "joint": the whole 4-component states are orthonormalised (BASELINE.json's literal recipe; config 0).
# "split": the u-pairs and the v-pairs are orthonormalised separately in their 2-component inner
#   products and recombined with the amplitudes sqrt(1-occ), sqrt(occ).  The set is then orthonormal in
#   the 4-component inner product as well (modified Gram-Schmidt leaves it unchanged) AND keeps the
#   particle number nwf*occ.  The joint recipe on thousands of u-dominated states pushes the weight of
#   the later states into v (measured: 1532 neutrons instead of 63 on config 1, 25x nuclear density,
#   far outside the ABM stability bound); DESIGN.md "input recipe".  Needs 2 * modes(kc) >= nwf:
#   kc raised to 2.0 (config 1) and 1.8 (config 2).
N_PEAK = (0.09, 0.07)  # fm^-3, neutron / proton peak densities (sum = saturation 0.16)


def occupancy(cfg, q, nwf_q):
    """v-component weight: literal for config 0, else scaled so the peak density is nuclear."""
    if cfg["occ"] is not None:
        return cfg["occ"][q]
    if nwf_q == 0:
        return 0.0
    occ = N_PEAK[q] * math.pi ** 1.5 * cfg["w"] ** 3 * len(cfg["centres"]) / nwf_q
    return min(occ, 0.5)


def _i64(x):
    x &= (1 << 64) - 1
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLD = _i64(0x9E3779B97F4A7C15)
_M1 = _i64(0xBF58476D1CE4E5B9)
_M2 = _i64(0x94D049BB133111EB)


def _lsr(x, s):
    return (x >> s) & ((1 << (64 - s)) - 1)


def _mix(z):
    """splitmix64 finaliser on int64 tensors (two's-complement wrap-around arithmetic)."""
    z = z + _GOLD
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    return z ^ _lsr(z, 31)


def _uniform_pm1(key, counter):
    """counter-based uniform(-1, 1): hash(key, counter) -> 53 random bits."""
    z = _mix(_mix(key) ^ (counter * _GOLD))
    return _lsr(z, 11).to(torch.float64) * (2.0 / (1 << 53)) - 1.0


def kgrid(shape, dx, device):
    """lattice wavevectors of PAPER.md Eq. 44 (only used to select |k| < kc modes)."""
    ks = []
    for n in shape:
        j = torch.arange(n, device=device, dtype=torch.float64)
        ks.append(torch.where(j < n / 2, j, j - n) * (2.0 * math.pi / (n * dx)))
    return torch.meshgrid(*ks, indexing="ij")


def envelope(shape, dx, w, centre, device):
    """periodised Gaussian of width w centred at box centre + `centre` (fm)."""
    env = torch.ones(shape, dtype=torch.float64, device=device)
    for ax, n in enumerate(shape):
        L = n * dx
        x = torch.arange(n, device=device, dtype=torch.float64) * dx
        c = 0.5 * L + centre[ax]
        e = torch.zeros(n, dtype=torch.float64, device=device)
        for m in range(-2, 3):
            e = e + torch.exp(-((x - c - m * L) ** 2) / (2.0 * w * w))
        view = [1, 1, 1]
        view[ax] = n
        env = env * e.view(view)
    return env


def raw_states(cfg, q, nwf_q, seed, device="cpu", first=0, count=None, scale=True):
    """un-orthonormalised states [count, 4, nx, ny, nz] complex128 (steps 1-3 of the recipe)."""
    shape, dx = cfg["shape"], cfg["dx"]
    count = nwf_q - first if count is None else count
    nxyz = shape[0] * shape[1] * shape[2]
    kx, ky, kz = kgrid(shape, dx, device)
    mask = ((kx * kx + ky * ky + kz * kz) < cfg["kc"] ** 2).to(torch.float64)
    occ = occupancy(cfg, q, nwf_q)
    amp = [math.sqrt(1.0 - occ)] * 2 + [math.sqrt(occ)] * 2
    mode = torch.arange(nxyz, device=device, dtype=torch.int64).view(shape)
    st = torch.arange(first, first + count, device=device, dtype=torch.int64).view(count, 1, 1, 1, 1)
    comp = torch.arange(4, device=device, dtype=torch.int64).view(1, 4, 1, 1, 1)
    out = torch.zeros((count, 4) + tuple(shape), dtype=torch.complex128, device=device)
    for ic, centre in enumerate(cfg["centres"]):
        key = (((seed * 2 + q) * (1 << 20) + st) * 4 + comp) * 8 + ic
        re = _uniform_pm1(key, 2 * mode)
        im = _uniform_pm1(key, 2 * mode + 1)
        coef = torch.complex(re * mask, im * mask)
        p = torch.fft.ifftn(coef, dim=(-3, -2, -1), norm="forward")   # sum_k a(k) e^{ik.r}
        out += p * envelope(shape, dx, cfg["w"], centre, device)
    if scale:
        for c in range(4):
            out[:, c] *= amp[c]
    return out


def orthonormalise(psi, dV):
    """Q factor (positive diagonal) of the states in <a|b> = dV sum conj(a) b, i.e. the result of
    modified Gram-Schmidt in state order, computed by Cholesky-QR applied three times (Householder QR
    if the Gram matrix is numerically singular)."""
    n = psi.shape[0]
    a = psi.reshape(n, -1)
    try:
        for _ in range(3):
            g = (a.conj() @ a.T) * dV          # g[k, l] = <k|l>
            g = 0.5 * (g + g.conj().T)
            L = torch.linalg.cholesky(g)       # g = L L^H
            # rows q_k = sum_l (conj(L)^-1)[k, l] a_l  (lower triangular: MGS order)
            a = torch.linalg.solve_triangular(L.conj(), a, upper=False)
    except Exception:
        qm, rm = torch.linalg.qr(psi.reshape(n, -1).T)            # columns = states
        d = torch.diagonal(rm)
        a = (qm * (d / d.abs()).conj().unsqueeze(0)).T.contiguous() / dV ** 0.5
    return a.reshape(psi.shape)


def make_species(cfg, q, nwf_q=None, seed=None, device="cpu", chunk=256):
    """orthonormal seeded states of species q: tensor [nwf_q, 4, nx, ny, nz] complex128."""
    nwf_q = cfg["nwf"][q] if nwf_q is None else nwf_q
    seed = SEED0 + CONFIGS.index(cfg) if seed is None else seed
    shape = tuple(cfg["shape"])
    if nwf_q == 0:
        return torch.zeros((0, 4) + shape, dtype=torch.complex128, device=device)
    return make_block(cfg, q, nwf_q, 0, nwf_q, seed, device, chunk)


def make_block(cfg, q, nwf_total, first, count, seed, device="cpu", chunk=256):
    """states [first, first+count) of a species with nwf_total states in all (the occupancy follows
    the total), orthonormalised within the block."""
    shape = tuple(cfg["shape"])
    dV = cfg["dx"] ** 3
    split = cfg.get("ortho", "joint") == "split"
    psi = torch.empty((count, 4) + shape, dtype=torch.complex128, device=device)
    for f in range(0, count, chunk):
        c = min(chunk, count - f)
        psi[f:f + c] = raw_states(cfg, q, nwf_total, seed, device, first=first + f, count=c, scale=not split)
    if not split:
        return orthonormalise(psi, dV)
    occ = occupancy(cfg, q, nwf_total)
    for half, amp in ((slice(0, 2), math.sqrt(1.0 - occ)), (slice(2, 4), math.sqrt(occ))):
        psi[:, half] = orthonormalise(psi[:, half].contiguous(), dV) * amp
    return psi


def make_config(idx, nwf=None, device="cpu"):
    """(cfg, [psi_n, psi_p]) for BASELINE config `idx`, optionally with reduced state counts."""
    cfg = CONFIGS[idx]
    nwf = cfg["nwf"] if nwf is None else nwf
    return cfg, [make_species(cfg, q, nwf[q], device=device) for q in (0, 1)]
