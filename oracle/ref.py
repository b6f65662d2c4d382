"""ctypes wrapper around the CPU oracle (oracle/lise_oracle.c).

TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It shares nothing with the CUDA path.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblise_oracle.so")
_SRC = os.path.join(_HERE, "lise_oracle.c")


def build(force=False):
    """Compile the oracle with gcc (-O2, OpenMP, no fast-math)."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= os.path.getmtime(_SRC)
            and os.path.getmtime(_SO) >= os.path.getmtime(os.path.join(_HERE, "lise_oracle.h"))):
        return _SO
    cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-Wall", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


class Params(C.Structure):
    _fields_ = ([(n, C.c_double) for n in
                 ("hbar2_2m", "e2", "hbarc", "t0", "t1", "t2", "t3", "x0", "x1", "x2", "x3", "gamma", "W0",
                  "g0_n", "g0_p")] + [(n, C.c_int) for n in ("coulomb", "pairing_rearrangement", "remove_phase")]
                + [(n, C.c_double) for n in ("alpha_pair", "mu_n", "mu_p", "e_cut")]
                + [(n, C.c_double * 3) for n in ("sea_a", "sea_b", "sea_c")]
                + [(n, C.c_double * 2) for n in ("sea_cdn", "sea_cdj")]
                + [(n, C.c_int) for n in ("functional", "pairing_cutoff", "renormalize")])


class ObservablesExt(C.Structure):
    _fields_ = ([(n, C.c_double * 3) for n in ("rcm", "rcm_n", "rcm_p")]
                + [(n, C.c_double) for n in ("q20", "q30", "q40")] + [("q21", C.c_double * 2), ("q22", C.c_double * 2)]
                + [(n, C.c_double) for n in ("delta_n", "delta_p", "e_coll")] + [("v_cm", C.c_double * 3)]
                + [(n, C.c_double) for n in ("e_cm", "e_ext")])

    def as_dict(self):
        out = {}
        for n, t in self._fields_:
            v = getattr(self, n)
            out[n] = v if isinstance(v, float) else list(v)
        return out


class Observables(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("energy", "e_kin", "e_skyrme", "e_coul", "e_pair", "n_neutron", "n_proton",
                 "norm_defect", "ortho_defect", "time")] + [("step", C.c_long)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.lise_ref_pairing_K.restype = C.c_double
        _lib.lise_ref_inv_geff_spherical.restype = C.c_double
        _lib.lise_ref_inv_geff_spherical.argtypes = [C.c_double] * 5
        _lib.lise_ref_set_time.argtypes = [C.c_void_p, C.c_double, C.c_long]
        _lib.lise_ref_set_external_amplitudes.argtypes = [C.c_void_p, C.c_double, C.c_double]
        _lib.lise_ref_abm_predict.argtypes = [C.c_long, C.c_double] + [C.c_void_p] * 9
        _lib.lise_ref_abm_correct.argtypes = [C.c_long, C.c_double] + [C.c_void_p] * 9
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle call {what} failed with code {rc}")


def default_params():
    p = Params()
    _chk(lib().lise_ref_default_params(C.byref(p)), "default_params")
    return p


def set_num_threads(n):
    return lib().lise_ref_set_num_threads(C.c_int(n))


def pairing_K():
    return lib().lise_ref_pairing_K()


def inv_geff_spherical(g0, M, U, mu, e_cut):
    return lib().lise_ref_inv_geff_spherical(g0, M, U, mu, e_cut)


def abm_predict(dt, y_n, y_nm1, f_n, f_nm1, f_nm2, f_nm3, e_n):
    arrs = [np.ascontiguousarray(a, dtype=np.complex128) for a in (y_n, y_nm1, f_n, f_nm1, f_nm2, f_nm3, e_n)]
    p = np.empty_like(arrs[0]); m = np.empty_like(arrs[0])
    _chk(lib().lise_ref_abm_predict(arrs[0].size, dt, *[_p(a) for a in arrs], _p(p), _p(m)), "abm_predict")
    return p, m


def abm_correct(dt, y_n, y_nm1, fm, f_n, f_nm1, f_nm2, p):
    arrs = [np.ascontiguousarray(a, dtype=np.complex128) for a in (y_n, y_nm1, fm, f_n, f_nm1, f_nm2, p)]
    y = np.empty_like(arrs[0]); e = np.empty_like(arrs[0])
    _chk(lib().lise_ref_abm_correct(arrs[0].size, dt, *[_p(a) for a in arrs], _p(y), _p(e)), "abm_correct")
    return y, e


class RefContext:
    """One oracle context (lattice, dt, state counts, wavefunctions and multistep history)."""

    def __init__(self, nx, ny, nz, dx, dt, nwf_n, nwf_p, params=None):
        self.shape = (nx, ny, nz)
        self.nxyz = nx * ny * nz
        self.dx, self.dt = dx, dt
        self.nwf = (nwf_n, nwf_p)
        self._h = C.c_void_p()
        _chk(lib().lise_ref_create(nx, ny, nz, C.c_double(dx), C.c_double(dt), nwf_n, nwf_p, C.byref(self._h)),
             "create")
        self.params = default_params()
        if nwf_p == 0:
            self.params.coulomb = 0
        if params is not None:
            self.set_params(params)

    def close(self):
        if self._h:
            lib().lise_ref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_params(self, params):
        self.params = params
        _chk(lib().lise_ref_set_params(self._h, C.byref(params)), "set_params")

    def set_dt(self, dt):
        self.dt = dt
        _chk(lib().lise_ref_set_dt(self._h, C.c_double(dt)), "set_dt")

    def set_time(self, time, step):
        _chk(lib().lise_ref_set_time(self._h, time, step), "set_time")

    def boost(self, q, chi):
        a = np.ascontiguousarray(chi, dtype=np.float64)
        assert a.size == self.nxyz
        _chk(lib().lise_ref_boost(self._h, q, _p(a)), "boost")

    def set_external_fields(self, q, u0=None, uvec=None):
        a = None if u0 is None else np.ascontiguousarray(u0, dtype=np.float64)
        b = None if uvec is None else np.ascontiguousarray(uvec, dtype=np.float64)
        assert a is None or a.size == self.nxyz
        assert b is None or b.size == 3 * self.nxyz
        _chk(lib().lise_ref_set_external_fields(self._h, q, None if a is None else _p(a), None if b is None else _p(b)),
             "set_external_fields")

    def set_external_amplitudes(self, f_now, f_next):
        _chk(lib().lise_ref_set_external_amplitudes(self._h, float(f_now), float(f_next)), "set_external_amplitudes")

    def set_frame(self, v_cm=(0, 0, 0), omega=(0, 0, 0), origin=(0, 0, 0)):
        arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (v_cm, omega, origin)]
        _chk(lib().lise_ref_set_frame(self._h, *[_p(a) for a in arrs]), "set_frame")

    def observables_ext(self):
        o = ObservablesExt()
        _chk(lib().lise_ref_observables_ext(self._h, C.byref(o)), "observables_ext")
        return o.as_dict()

    def moments_from(self, dens_n, dens_p, pot_n, pot_p):
        arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (dens_n, dens_p, pot_n, pot_p)]
        o = ObservablesExt()
        _chk(lib().lise_ref_moments_from(self._h, *[_p(a) for a in arrs], C.byref(o)), "moments_from")
        return o.as_dict()

    def _blk(self, q, a):
        a = np.ascontiguousarray(a, dtype=np.complex128)
        assert a.size == self.nwf[q] * 4 * self.nxyz, (a.shape, self.nwf[q], self.nxyz)
        return a

    def set_wavefunctions(self, q, psi):
        a = self._blk(q, psi)
        _chk(lib().lise_ref_set_wavefunctions(self._h, q, _p(a)), "set_wavefunctions")

    def get_wavefunctions(self, q):
        out = np.empty((self.nwf[q], 4) + self.shape, dtype=np.complex128)
        _chk(lib().lise_ref_get_wavefunctions(self._h, q, _p(out)), "get_wavefunctions")
        return out

    def set_history(self, q, y_nm1, f_nm1, f_nm2, f_nm3, e_n):
        arrs = [self._blk(q, a) for a in (y_nm1, f_nm1, f_nm2, f_nm3, e_n)]
        _chk(lib().lise_ref_set_history(self._h, q, *[_p(a) for a in arrs]), "set_history")

    def densities(self, q):
        out = np.empty((14,) + self.shape)
        _chk(lib().lise_ref_densities(self._h, q, _p(out)), "densities")
        return out

    def densities_of(self, psi):
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        nst = a.size // (4 * self.nxyz)
        out = np.empty((14,) + self.shape)
        _chk(lib().lise_ref_densities_of(self._h, _p(a), nst, _p(out)), "densities_of")
        return out

    def potentials(self, q):
        out = np.empty((14,) + self.shape)
        _chk(lib().lise_ref_potentials(self._h, q, _p(out)), "potentials")
        return out

    def potentials_from(self, dens_n, dens_p):
        dn = np.ascontiguousarray(dens_n, dtype=np.float64); dp = np.ascontiguousarray(dens_p, dtype=np.float64)
        pn = np.empty((14,) + self.shape); pp = np.empty((14,) + self.shape)
        e5 = np.zeros(5)
        _chk(lib().lise_ref_potentials_from(self._h, _p(dn), _p(dp), _p(pn), _p(pp), _p(e5)), "potentials_from")
        return pn, pp, e5

    def apply_h(self, q, psi):
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        nst = a.size // (4 * self.nxyz)
        out = np.empty_like(a)
        _chk(lib().lise_ref_apply_h(self._h, q, _p(a), _p(out), nst), "apply_h")
        return out

    def apply_h_with(self, pot14, psi):
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        pot = np.ascontiguousarray(pot14, dtype=np.float64)
        nst = a.size // (4 * self.nxyz)
        out = np.empty_like(a)
        _chk(lib().lise_ref_apply_h_with(self._h, _p(pot), _p(a), _p(out), nst), "apply_h_with")
        return out

    def step(self, nsteps):
        _chk(lib().lise_ref_step(self._h, nsteps), "step")

    def observables(self):
        o = Observables()
        _chk(lib().lise_ref_observables(self._h, C.byref(o)), "observables")
        return o.as_dict()

    def deriv_matrix(self, axis, order):
        n = self.shape[axis]
        out = np.empty((n, n))
        _chk(lib().lise_ref_deriv_matrix(self._h, axis, order, _p(out)), "deriv_matrix")
        return out

    def deriv(self, axis, order, fields):
        a = np.ascontiguousarray(fields, dtype=np.complex128)
        nf = a.size // self.nxyz
        out = np.empty_like(a)
        _chk(lib().lise_ref_deriv(self._h, axis, order, _p(a), _p(out), nf), "deriv")
        return out

    def coulomb(self, n_p):
        a = np.ascontiguousarray(n_p, dtype=np.float64)
        out = np.empty(self.shape)
        _chk(lib().lise_ref_coulomb(self._h, _p(a), _p(out)), "coulomb")
        return out
