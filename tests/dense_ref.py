"""Brute-force numpy constructions used ONLY to pin the oracle (never by the product path).

Written from PAPER.md independently of oracle/lise_oracle.c: the DVR derivative matrices in their
closed forms (Eq. 48a, and Eq. 48b with the corrected off-diagonal prefactor, reading B3),
Kronecker products for 3D, explicit operator products and the block structure of Eq. 11.
"""
import numpy as np

SIG = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]], complex)]


def eps(i, j, k):
    return (i - j) * (j - k) * (k - i) // 2


def dvr_d1(N, a):
    """PAPER.md Eq. 48a: (d/dx)_{nm} = (pi/(N a)) (-1)^{n-m} cot(pi (n-m)/N), 0 on the diagonal."""
    D = np.zeros((N, N))
    for n in range(N):
        for m in range(N):
            if n != m:
                D[n, m] = np.pi / (N * a) * (-1.0) ** (n - m) / np.tan(np.pi * (n - m) / N)
    return D


def dvr_d2(N, a):
    """PAPER.md Eq. 48b with the off-diagonal prefactor 2 pi^2/(N^2 a^2) (printed: pi^2/(2 N^2 a^2))."""
    D = np.zeros((N, N))
    for n in range(N):
        for m in range(N):
            if n != m:
                D[n, m] = 2.0 * np.pi ** 2 / (N * N * a * a) * (-1.0) ** (n - m + 1) / np.sin(np.pi * (n - m) / N) ** 2
            else:
                D[n, m] = -np.pi ** 2 / (3.0 * a * a) * (1.0 + 2.0 / (N * N))
    return D


def kron3(mats, shape, axis):
    """operator acting with `mats` along `axis` of a [nx][ny][nz] (iz fastest) lattice."""
    ops = [np.eye(n) for n in shape]
    ops[axis] = mats
    return np.kron(np.kron(ops[0], ops[1]), ops[2])


def dense_h(shape, a, pot):
    """single-particle h (2 Nxyz x 2 Nxyz, spin-major) of PAPER.md Eq. 12 in the adopted lattice form
    (Eqs. 55, 56, operator-product current term).  pot: dict U, M, W[3], S[3], A[3] (flat real arrays)."""
    nxyz = int(np.prod(shape))
    D = [kron3(dvr_d1(shape[i], a), shape, i) for i in range(3)]
    L = sum(kron3(dvr_d2(shape[i], a), shape, i) for i in range(3))
    dg = np.diag
    M, U = pot["M"], pot["U"]
    lapM = L @ M
    h0 = -0.5 * (dg(M) @ L + L @ dg(M)) + 0.5 * dg(lapM) + dg(U)
    for i in range(3):
        h0 = h0 - 1j * (dg(pot["A"][i]) @ D[i] + D[i] @ dg(pot["A"][i]))
    h = np.kron(np.eye(2), h0).astype(complex)
    for m in range(3):
        h += np.kron(SIG[m], dg(pot["S"][m]))
    for i in range(3):
        for j in range(3):
            for k in range(3):
                e = eps(i, j, k)
                if e:
                    h += -0.5j * e * np.kron(SIG[j], dg(pot["W"][k]) @ D[i] + D[i] @ dg(pot["W"][k]))
    return h


def dense_H(shape, a, pot):
    """quasiparticle Hamiltonian of PAPER.md Eq. 11 with mu = 0; basis order (u_up, u_dn, v_up, v_dn)."""
    nxyz = int(np.prod(shape))
    h = dense_h(shape, a, pot)
    Dl = np.diag(pot["Delta"])
    Z = np.zeros((nxyz, nxyz), complex)
    ur = np.block([[Z, Dl], [-Dl, Z]])
    ll = np.block([[Z, -Dl.conj()], [Dl.conj(), Z]])
    return np.block([[h, ur], [ll, -h.conj()]])


def random_potentials(shape, rng, smooth=True):
    """random real potential fields (flat) and the Table-3 array [14, nx, ny, nz] the oracle takes."""
    nxyz = int(np.prod(shape))

    def fld():
        f = rng.standard_normal(shape)
        if smooth:
            fk = np.fft.fftn(f)
            k = np.meshgrid(*[np.fft.fftfreq(n) * n for n in shape], indexing="ij")
            fk *= np.exp(-0.5 * sum(q * q for q in k))
            f = np.real(np.fft.ifftn(fk))
        return f.reshape(-1)

    pot = dict(U=30 * fld(), M=20.7 + 8 * np.abs(fld()), W=[10 * fld() for _ in range(3)],
               S=[5 * fld() for _ in range(3)], A=[4 * fld() for _ in range(3)],
               Delta=3 * (fld() + 1j * fld()))
    return pot


def table3(pot, lapM, shape):
    t = np.zeros((14,) + tuple(shape))
    t[0] = pot["U"].reshape(shape); t[1] = pot["M"].reshape(shape); t[2] = lapM.reshape(shape)
    for i in range(3):
        t[3 + i] = pot["W"][i].reshape(shape)
        t[6 + i] = pot["S"][i].reshape(shape)
        t[9 + i] = pot["A"][i].reshape(shape)
    t[12] = pot["Delta"].real.reshape(shape); t[13] = pot["Delta"].imag.reshape(shape)
    return t


def scf_ground_state(c, shape, a, nocc=2, width=1.8, mix=0.5, tol=1e-13, maxit=400):
    """Self-consistent Hartree-Fock state in the mean field of the oracle context `c` (pairing must be off): per species
    the `nocc` lowest orbitals of the dense single-particle h (dense_h above) occupied as v_k = conj(phi_k), u_k = 0
    (Eq. 11: the v sector carries -h*), iterated with linear mixing of the 14 density fields until they stop changing.
    Returns (psi[2] as [nocc, 4, nx, ny, nz] complex, eps[2] single-particle energies, iterations, last change)."""
    import math
    nxyz = int(np.prod(shape)); dV = a ** 3
    x = np.meshgrid(*[(np.arange(n) - n / 2 + 0.5) * a for n in shape], indexing="ij")
    g = np.exp(-sum(q * q for q in x) / (2 * width ** 2)); g /= math.sqrt(dV * (g * g).sum())

    def states(orbs):                       # [nocc, 2 nxyz] spin-major spinors phi_k -> psi_k = (0, 0, conj phi_k)
        psi = np.zeros((nocc, 4) + tuple(shape), complex)
        for k in range(nocc):
            psi[k, 2:] = np.conj(orbs[k]).reshape((2,) + tuple(shape))
        return psi
    orb0 = np.zeros((nocc, 2 * nxyz), complex)
    for k in range(nocc):
        orb0[k, (k % 2) * nxyz:(k % 2 + 1) * nxyz] = g.reshape(-1) * (1.0 + 0.1 * (k // 2) * x[0].reshape(-1))
    psi = [states(orb0), states(orb0)]
    dens = [c.densities_of(p) for p in psi]
    eps = [None, None]
    change = None
    for it in range(maxit):
        pn, pp, _ = c.potentials_from(dens[0], dens[1])
        for q, t in enumerate((pn, pp)):
            pot = dict(U=t[0].reshape(-1), M=t[1].reshape(-1), W=[t[3 + i].reshape(-1) for i in range(3)],
                       S=[t[6 + i].reshape(-1) for i in range(3)], A=[t[9 + i].reshape(-1) for i in range(3)])
            h = dense_h(shape, a, pot)
            assert np.abs(h - h.conj().T).max() < 1e-9
            w, v = np.linalg.eigh(h)
            eps[q] = w[:nocc]
            psi[q] = states((v[:, :nocc] / math.sqrt(dV)).T)
        new = [c.densities_of(p) for p in psi]
        change = max(np.abs(n_ - d_).max() for n_, d_ in zip(new, dens))
        dens = [(1.0 - mix) * d_ + mix * n_ for n_, d_ in zip(new, dens)]
        if change < tol:
            break
    return psi, eps, it, change
