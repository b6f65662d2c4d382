"""Host logic of the CUDA library that needs no GPU: the block-diagonalised line-operator tables
(include/lise.h: lise_line_operator_tables) applied in numpy must reproduce the FFT
derivative of PAPER.md Eqs. 49-50 (L403-L412: ik with the Nyquist mode zeroed, -k^2 with it kept)."""
import numpy as np
import pytest

from paper_2009_00745_b200 import lise


def fft_derivatives(x, dx):
    n = x.shape[0]
    k = 2.0 * np.pi * np.fft.fftfreq(n, d=dx)
    k1 = k.copy(); k1[n // 2] = 0.0
    xh = np.fft.fft(x)
    return np.fft.ifft(1j * k1 * xh), np.fft.ifft(-(k ** 2) * xh)


def apply_tables(dims, tab, op, x):
    """the algorithm of split_lineop.cuh written out with plain loops"""
    H, R, J, ND = dims["H"], dims["R"], dims["J"], dims["ND"]
    xs = x.reshape(R, H)
    y = np.zeros((R, H), dtype=x.dtype)
    for j in range(J):
        if j > 0 and 2 * j != R and j > (R - 1) // 2:
            continue
        cos = np.cos(2 * np.pi * j * np.arange(R) / R); sin = np.sin(2 * np.pi * j * np.arange(R) / R)
        b = (cos[:, None] * xs).sum(0); e = (sin[:, None] * xs).sum(0)
        P = np.array([[tab[op, j, 0, r - rp + H - 1] for rp in range(H)] for r in range(H)])
        Q = np.array([[tab[op, j, 1, r - rp + H - 1] for rp in range(H)] for r in range(H)])
        S = P @ b - Q @ e; T = P @ e + Q @ b
        y += cos[:, None] * S[None, :] + sin[:, None] * T[None, :]
    return y.reshape(-1)


@pytest.mark.parametrize("n", [8, 12, 16, 20, 24, 32, 40, 48, 64])
def test_block_diagonalised_tables_reproduce_fft_derivatives(n):
    dx = 1.25
    dims, tab = lise.line_operator_tables(n, dx)
    assert dims["H"] * dims["R"] == n
    assert dims["H"] == (8 if n % 8 == 0 and n >= 16 else n)
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    d1, d2 = fft_derivatives(x, dx)
    g1 = apply_tables(dims, tab, 0, x); g2 = apply_tables(dims, tab, 1, x)
    assert np.abs(g1 - d1).max() <= 2e-13 * np.abs(d1).max()
    assert np.abs(g2 - d2).max() <= 2e-13 * np.abs(d2).max()


def test_tables_reject_bad_arguments():
    lib = lise.load()
    import ctypes as C
    dims = (C.c_int * 5)()
    assert lib.lise_line_operator_tables(10, 1.0, None, 0, dims) != 0      # n % 4 != 0
    assert lib.lise_line_operator_tables(16, -1.0, None, 0, dims) != 0
    assert lib.lise_line_operator_tables(16, 1.0, None, 0, dims) == 0
    buf = (C.c_double * 4)()
    assert lib.lise_line_operator_tables(16, 1.0, buf, 4, dims) != 0       # capacity too small


def test_capacity_states_never_returns_more_than_fits():
    """7 state arrays of 64 Nxyz bytes per state + a reserve must fit the free memory."""
    from paper_2009_00745_b200 import lise
    shape = (32, 32, 32); S = 64 * 32 ** 3; G = 2 ** 30
    fits = lambda nwf, free, reserve: 7 * S * sum(nwf) + reserve <= free
    assert lise.capacity_states(shape, 180 * G, (4096, 4096)) == (4096, 4096)          # the request fits: unchanged
    got = lise.capacity_states(shape, 180 * G, (8192, 8192))                            # SURVEY finding 5: 16384 do not
    assert got[0] == got[1] and got[0] % 256 == 0 and 0 < got[0] < 8192 and fits(got, 180 * G, 6 * G)
    assert not fits((got[0] + 256, got[1] + 256), 180 * G, 6 * G)                       # and it is the largest such count
    got = lise.capacity_states(shape, 100 * G, (12000, 0))                              # one species gets the whole device
    assert got[1] == 0 and got[0] % 256 == 0 and got[0] > 6000 and fits(got, 100 * G, 6 * G)
    got = lise.capacity_states(shape, 100 * G, (9000, 3000))                            # split follows the request
    assert fits(got, 100 * G, 6 * G) and 2.5 < got[0] / got[1] < 3.5
    assert lise.capacity_states(shape, 6 * G + 7 * S * 300, (4096, 4096)) == (0, 0)     # under 256 per species: nothing
    assert lise.capacity_states(shape, 2 * G, (4096, 4096)) == (0, 0)                   # less free than the reserve
    assert lise.capacity_states(shape, 2 * G, (0, 0)) == (0, 0)
