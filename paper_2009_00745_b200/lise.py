"""Thin ctypes binding of liblise.so (include/lise.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; torch is used for device memory and
streams.  There is no CPU fallback: if the library is missing or no CUDA device is present, calls fail.
"""
import ctypes as C
import os

import torch

from . import build as _build

_lib = None


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
        for n, _ in self._fields_:
            v = getattr(self, n)
            out[n] = v if isinstance(v, float) else list(v)
        return out


class Observables(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("energy", "e_kin", "e_skyrme", "e_coul", "e_pair", "n_neutron", "n_proton",
                 "norm_defect", "ortho_defect", "time")] + [("step", C.c_long)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


EXPORTS = ["lise_default_params", "lise_create", "lise_destroy", "lise_set_params", "lise_set_stream",
           "lise_set_dt", "lise_set_chunk", "lise_set_overlap", "lise_set_wavefunctions", "lise_get_wavefunctions",
           "lise_upload_wavefunctions", "lise_download_wavefunctions", "lise_set_reduce_hook",
           "lise_densities", "lise_potentials", "lise_apply_h", "lise_step", "lise_observables", "lise_observables_ext",
           "lise_set_time", "lise_boost", "lise_set_external_fields", "lise_set_frame",
           "lise_profile", "lise_profile_read", "lise_measure_fp64_peak", "lise_set_density_group", "lise_line_operator", "lise_line_operator_cost", "lise_line_operator_tables", "lise_launch_count", "lise_device_bytes", "lise_strerror", "lise_last_error",
           "lise_renormalize_static", "lise_static_last_error", "lise_create_with_line_operator",
           "lise_set_external_amplitudes"]

STATIC_MAX_STATES = 16384       # LISE_STATIC_MAX_STATES of include/lise.h


REDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_long)


class _DevView:
    """__cuda_array_interface__ wrapper of a raw device pointer (float64), for torch.as_tensor."""

    def __init__(self, ptr, count):
        self.__cuda_array_interface__ = {"shape": (count,), "typestr": "<f8", "data": (ptr, False), "version": 3,
                                         "strides": None}


def lib_path():
    return _build.SO


def load():
    """dlopen the in-tree liblise.so (building it with nvcc if the sources are newer)."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        _build.build()          # serialised across processes by a file lock; written to a temp file, then renamed
    except Exception as exc:  # nvcc missing on the box: use the shipped .so if there is one
        if not os.path.exists(_build.SO):
            raise RuntimeError(f"liblise.so is missing and could not be built: {exc}") from exc
    lib = C.CDLL(_build.SO)
    vp, ip, dp = C.c_void_p, C.c_int, C.c_double
    lib.lise_default_params.argtypes = [C.POINTER(Params)]
    lib.lise_create.argtypes = [ip, ip, ip, dp, dp, ip, ip, C.POINTER(vp)]
    lib.lise_create_with_line_operator.argtypes = [ip, ip, ip, dp, dp, ip, ip, C.c_char_p, C.POINTER(vp)]
    lib.lise_destroy.argtypes = [vp]; lib.lise_destroy.restype = None
    lib.lise_set_params.argtypes = [vp, C.POINTER(Params)]
    lib.lise_set_stream.argtypes = [vp, vp]
    lib.lise_set_dt.argtypes = [vp, dp]
    lib.lise_set_chunk.argtypes = [vp, ip]
    lib.lise_set_overlap.argtypes = [vp, ip]
    lib.lise_set_wavefunctions.argtypes = [vp, ip, vp]
    lib.lise_get_wavefunctions.argtypes = [vp, ip, vp]
    lib.lise_upload_wavefunctions.argtypes = [vp, ip, vp, ip]
    lib.lise_download_wavefunctions.argtypes = [vp, ip, vp]
    lib.lise_set_reduce_hook.argtypes = [vp, REDUCE_FN, vp]
    lib.lise_densities.argtypes = [vp, ip, vp]
    lib.lise_potentials.argtypes = [vp, ip, vp]
    lib.lise_apply_h.argtypes = [vp, ip, vp, vp, ip]
    lib.lise_step.argtypes = [vp, ip]
    lib.lise_observables.argtypes = [vp, C.POINTER(Observables)]
    lib.lise_observables_ext.argtypes = [vp, C.POINTER(ObservablesExt)]
    lib.lise_set_time.argtypes = [vp, dp, C.c_long]
    lib.lise_boost.argtypes = [vp, ip, vp]
    lib.lise_set_external_fields.argtypes = [vp, ip, vp, vp]
    lib.lise_set_frame.argtypes = [vp, C.POINTER(dp), C.POINTER(dp), C.POINTER(dp)]
    lib.lise_set_external_amplitudes.argtypes = [vp, dp, dp]
    lib.lise_profile.argtypes = [vp, ip]
    lib.lise_profile_read.argtypes = [vp, C.POINTER(dp), C.POINTER(C.c_long)]
    lib.lise_measure_fp64_peak.argtypes = [vp, dp, C.POINTER(dp), C.POINTER(dp)]
    lib.lise_line_operator.argtypes = [vp]; lib.lise_line_operator.restype = C.c_char_p
    lib.lise_set_density_group.argtypes = [vp, ip]
    lib.lise_line_operator_cost.argtypes = [ip, C.POINTER(ip), C.POINTER(ip)]
    lib.lise_line_operator_tables.argtypes = [ip, dp, C.POINTER(dp), ip, C.POINTER(ip)]
    lib.lise_launch_count.argtypes = [vp]; lib.lise_launch_count.restype = C.c_long
    lib.lise_device_bytes.argtypes = [vp]; lib.lise_device_bytes.restype = C.c_longlong
    lib.lise_strerror.argtypes = [ip]; lib.lise_strerror.restype = C.c_char_p
    lib.lise_last_error.argtypes = [vp]; lib.lise_last_error.restype = C.c_char_p
    lib.lise_renormalize_static.argtypes = [vp, ip, C.c_longlong, dp, vp]
    lib.lise_static_last_error.argtypes = []; lib.lise_static_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def default_params():
    p = Params()
    load().lise_default_params(C.byref(p))
    return p


def measure_fp64_peak(seconds=1.0, stream=None):
    """sustained fp64 FMA throughput of the current device in TFLOP/s (DFMA microbenchmark)."""
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device")
    st = torch.cuda.current_stream() if stream is None else stream
    tf = C.c_double(); mhz = C.c_double()
    rc = load().lise_measure_fp64_peak(C.c_void_p(st.cuda_stream), seconds, C.byref(tf), C.byref(mhz))
    if rc != 0:
        raise RuntimeError(f"lise_measure_fp64_peak failed ({rc})")
    return tf.value


def renormalize_static(psi, dV, stream=None):
    """lise_renormalize_static: psi[k] <- psi[k] / sqrt(dV sum |psi[k]|^2) in place, for a contiguous CUDA complex128
    tensor whose first axis counts the states (at most STATIC_MAX_STATES of them).  For callers that cannot let the
    library allocate device memory (HBM already full of wavefunctions, or no cudaMalloc stall allowed in the time
    loop): no context, and the per-state scratch is a fixed array inside liblise.so, shared by all calls on a device --
    calls that may overlap on the GPU must be ordered by the caller.  Enqueued on `stream` (default: torch's current
    stream on psi's device); does not synchronise."""
    if not (psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.dim() >= 2):
        raise LiseError("renormalize_static expects a contiguous CUDA complex128 tensor [nstates, ...]")
    lib = load()
    nst = psi.shape[0]
    slen = psi.numel() // nst if nst else 1
    with torch.cuda.device(psi.device):
        st = torch.cuda.current_stream(psi.device) if stream is None else stream
        rc = lib.lise_renormalize_static(C.c_void_p(psi.data_ptr()), nst, slen, float(dV), C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise LiseError(f"lise_renormalize_static failed: {lib.lise_strerror(rc).decode()} ({rc}) "
                        f"{lib.lise_static_last_error().decode()}")
    return psi


def line_operator_cost(n):
    """(inner, outer) fp64 instruction counts of the generated FFT code for a real line of n points; host only."""
    a, b = C.c_int(), C.c_int()
    rc = load().lise_line_operator_cost(n, C.byref(a), C.byref(b))
    if rc != 0:
        raise RuntimeError(f"lise_line_operator_cost failed ({rc})")
    return a.value, b.value


def line_operator_tables(n, dx):
    """(dims dict, table as a numpy array [op][j][P|Q][d]) of the block-diagonalised line operator; host only."""
    import numpy as np
    lib = load()
    dims = (C.c_int * 5)()
    rc = lib.lise_line_operator_tables(n, dx, None, 0, dims)
    if rc != 0:
        raise RuntimeError(f"lise_line_operator_tables: {lib.lise_strerror(rc).decode()}")
    H, R, J, ND, size = (int(v) for v in dims)
    tab = np.zeros(size, dtype=np.float64)
    rc = lib.lise_line_operator_tables(n, dx, tab.ctypes.data_as(C.POINTER(C.c_double)), size, dims)
    if rc != 0:
        raise RuntimeError(f"lise_line_operator_tables: {lib.lise_strerror(rc).decode()}")
    return dict(H=H, R=R, J=J, ND=ND), tab.reshape(2, J, 2, ND)


def capacity_states(shape, free_bytes, requested, reserve_bytes=6 * 2 ** 30, multiple=256):
    """capacity rule of SURVEY 8(d) / Appendix C: the library keeps 7 state arrays of S = 64 Nxyz bytes per state
    (+ a chunk-sized H psi scratch and grid fields, covered by `reserve_bytes`).  Returns the (n, p) state counts that
    fit `free_bytes` of device memory: `requested` if it fits; else the capacity split in proportion to the request,
    each species rounded down to a multiple of `multiple`; (0, 0) if that leaves a requested species without states
    (the workload does not fit: the caller skips it instead of running into an out-of-memory error in lise_create)."""
    S = 64 * shape[0] * shape[1] * shape[2]
    cap = max(0, int((free_bytes - reserve_bytes) // (7 * S)))
    req = (int(requested[0]), int(requested[1]))
    tot = req[0] + req[1]
    if tot <= cap:
        return req
    fit = tuple(min(r, (cap * r // tot) // multiple * multiple) for r in req)
    if any(r > 0 and f == 0 for r, f in zip(req, fit)):
        return (0, 0)
    return fit


class LiseError(RuntimeError):
    pass


class Lise:
    """One TDSLDA context on the current CUDA device.  Tensors are torch CUDA tensors (complex128 / float64)."""

    def __init__(self, nx, ny, nz, dx, dt, nwf_n, nwf_p, params=None, stream=None, device=None, line_operator=None):
        if not torch.cuda.is_available():
            raise LiseError("no CUDA device: the TDSLDA path has no CPU fallback")
        self.lib = load()
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.shape = (nx, ny, nz)
        self.nxyz = nx * ny * nz
        self.nwf = (nwf_n, nwf_p)
        self.dx, self.dt = dx, dt
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            if line_operator is None:
                rc = self.lib.lise_create(nx, ny, nz, dx, dt, nwf_n, nwf_p, C.byref(self._h))
            else:       # "fft" | "dmma" | "dense" | "auto": lise_create_with_line_operator
                rc = self.lib.lise_create_with_line_operator(nx, ny, nz, dx, dt, nwf_n, nwf_p, line_operator.encode(), C.byref(self._h))
        if rc != 0:
            self._h = C.c_void_p()
            raise LiseError(f"lise_create failed: {self.lib.lise_strerror(rc).decode()} ({rc}) {self.lib.lise_last_error(None).decode()}")
        st = torch.cuda.current_stream(self.device) if stream is None else stream
        self._stream_ptr = st.cuda_stream
        self._chk(self.lib.lise_set_stream(self._h, C.c_void_p(st.cuda_stream)), "lise_set_stream")
        self.params = default_params()
        self.coulomb_requested = int(self.params.coulomb)   # what the caller asked for (sharding.attach decides from it)
        if nwf_p == 0:
            self.params.coulomb = 0            # lise_create's default for a context without proton states
        if params is not None:
            self.set_params(params)

    def _chk(self, rc, what):
        if rc != 0 and getattr(self, "_hook_error", None) is not None:
            exc, self._hook_error = self._hook_error, None
            raise LiseError(f"{what} failed in the reduce hook: {exc!r}") from exc
        if rc != 0:
            msg = self.lib.lise_last_error(self._h).decode() if self._h else ""
            raise LiseError(f"{what} failed: {self.lib.lise_strerror(rc).decode()} ({rc}) {msg}")

    def close(self):
        if getattr(self, "_h", None):
            self.lib.lise_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, t, dtype, numel):
        if not (t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.numel() == numel):
            raise LiseError(f"expected a contiguous CUDA {dtype} tensor with {numel} elements, got "
                            f"{t.dtype} {tuple(t.shape)} on {t.device}")
        return C.c_void_p(t.data_ptr())

    def set_params(self, params):
        self.params = params
        self.coulomb_requested = int(params.coulomb)
        self._chk(self.lib.lise_set_params(self._h, C.byref(params)), "lise_set_params")

    def set_stream(self, stream):
        self._stream_ptr = stream.cuda_stream
        self._chk(self.lib.lise_set_stream(self._h, C.c_void_p(stream.cuda_stream)), "lise_set_stream")

    def set_density_group(self, nchunks):
        self._chk(self.lib.lise_set_density_group(self._h, nchunks), "lise_set_density_group")

    def set_dt(self, dt):
        self.dt = dt
        self._chk(self.lib.lise_set_dt(self._h, dt), "lise_set_dt")

    def set_chunk(self, n):
        self._chk(self.lib.lise_set_chunk(self._h, n), "lise_set_chunk")

    def set_overlap(self, enable):
        self._chk(self.lib.lise_set_overlap(self._h, int(enable)), "lise_set_overlap")

    def set_wavefunctions(self, q, psi):
        p = self._dev(psi, torch.complex128, self.nwf[q] * 4 * self.nxyz) if self.nwf[q] else C.c_void_p()
        self._chk(self.lib.lise_set_wavefunctions(self._h, q, p), "lise_set_wavefunctions")

    def get_wavefunctions(self, q, out=None):
        if out is None:
            out = torch.empty((self.nwf[q], 4) + self.shape, dtype=torch.complex128, device=self.device)
        p = self._dev(out, torch.complex128, self.nwf[q] * 4 * self.nxyz) if self.nwf[q] else C.c_void_p()
        self._chk(self.lib.lise_get_wavefunctions(self._h, q, p), "lise_get_wavefunctions")
        return out

    def _host(self, t, numel):
        if not (t.device.type == "cpu" and t.dtype == torch.complex128 and t.is_contiguous() and t.numel() == numel):
            raise LiseError(f"expected a contiguous CPU complex128 tensor with {numel} elements")
        return C.c_void_p(t.data_ptr())

    def upload_wavefunctions(self, q, psi_host, keep_history=False):
        """host tensor (pinned for speed) -> y_n of species q, through the library's own H2D copy."""
        p = self._host(psi_host, self.nwf[q] * 4 * self.nxyz) if self.nwf[q] else C.c_void_p()
        self._chk(self.lib.lise_upload_wavefunctions(self._h, q, p, int(keep_history)), "lise_upload_wavefunctions")

    def download_wavefunctions(self, q, out_host):
        p = self._host(out_host, self.nwf[q] * 4 * self.nxyz) if self.nwf[q] else C.c_void_p()
        self._chk(self.lib.lise_download_wavefunctions(self._h, q, p), "lise_download_wavefunctions")
        return out_host

    def set_reduce_hook(self, reduce_tensor):
        """reduce_tensor(t): in-place sum over ranks of the float64 CUDA tensor t, enqueued on the
        context's stream (e.g. lambda t: torch.distributed.all_reduce(t)).  None removes the hook."""
        if reduce_tensor is None:
            self._hook = None
            self._chk(self.lib.lise_set_reduce_hook(self._h, REDUCE_FN(0), None), "lise_set_reduce_hook")
            return

        def _cb(user, ptr, count):
            try:
                # lise.h: the reduction must be enqueued on the CONTEXT's stream, which need not be torch's current one
                with torch.cuda.device(self.device), torch.cuda.stream(torch.cuda.ExternalStream(self._stream_ptr, device=self.device)):
                    reduce_tensor(torch.as_tensor(_DevView(ptr, count), device=self.device))
                return 0
            except Exception as exc:  # never let an exception cross the C ABI
                self._hook_error = exc
                return 1
        self._hook = REDUCE_FN(_cb)     # keep alive
        self._chk(self.lib.lise_set_reduce_hook(self._h, self._hook, None), "lise_set_reduce_hook")

    def densities(self, q, out=None):
        if out is None:
            out = torch.empty((14,) + self.shape, dtype=torch.float64, device=self.device)
        self._chk(self.lib.lise_densities(self._h, q, self._dev(out, torch.float64, 14 * self.nxyz)), "lise_densities")
        return out

    def potentials(self, q, out=None):
        if out is None:
            out = torch.empty((14,) + self.shape, dtype=torch.float64, device=self.device)
        self._chk(self.lib.lise_potentials(self._h, q, self._dev(out, torch.float64, 14 * self.nxyz)), "lise_potentials")
        return out

    def apply_h(self, q, psi, out=None):
        nst = psi.numel() // (4 * self.nxyz)
        if out is None:
            out = torch.empty_like(psi)
        self._chk(self.lib.lise_apply_h(self._h, q, self._dev(psi, torch.complex128, nst * 4 * self.nxyz),
                                        self._dev(out, torch.complex128, nst * 4 * self.nxyz), nst), "lise_apply_h")
        return out

    def step(self, nsteps=1):
        self._chk(self.lib.lise_step(self._h, nsteps), "lise_step")

    def observables(self):
        o = Observables()
        self._chk(self.lib.lise_observables(self._h, C.byref(o)), "lise_observables")
        return o.as_dict()

    def observables_ext(self):
        o = ObservablesExt()
        self._chk(self.lib.lise_observables_ext(self._h, C.byref(o)), "lise_observables_ext")
        return o.as_dict()

    def set_time(self, time, step):
        self._chk(self.lib.lise_set_time(self._h, time, step), "lise_set_time")

    def boost(self, q, chi):
        self._chk(self.lib.lise_boost(self._h, q, self._dev(chi, torch.float64, self.nxyz)), "lise_boost")

    def set_external_fields(self, q, u0=None, uvec=None):
        a = C.c_void_p() if u0 is None else self._dev(u0, torch.float64, self.nxyz)
        b = C.c_void_p() if uvec is None else self._dev(uvec, torch.float64, 3 * self.nxyz)
        self._chk(self.lib.lise_set_external_fields(self._h, q, a, b), "lise_set_external_fields")

    def set_external_amplitudes(self, f_now, f_next):
        """f(t_n), f(t_n + dt) on the profiles of set_external_fields; call before every step(1) of a driven run."""
        self._chk(self.lib.lise_set_external_amplitudes(self._h, float(f_now), float(f_next)), "lise_set_external_amplitudes")

    def set_frame(self, v_cm=(0.0, 0.0, 0.0), omega=(0.0, 0.0, 0.0), origin=(0.0, 0.0, 0.0)):
        arrs = [(C.c_double * 3)(*[float(x) for x in v]) for v in (v_cm, omega, origin)]
        self._chk(self.lib.lise_set_frame(self._h, *arrs), "lise_set_frame")

    PROFILE_CLASSES = ("happly_yz", "happly_xz", "update", "dens_x", "grid", "dens_yz")

    def profile(self, enable=True):
        self._chk(self.lib.lise_profile(self._h, int(enable)), "lise_profile")

    def profile_read(self):
        ms = (C.c_double * 6)(); cnt = (C.c_long * 6)()
        self._chk(self.lib.lise_profile_read(self._h, ms, cnt), "lise_profile_read")
        return {n: (ms[i], cnt[i]) for i, n in enumerate(self.PROFILE_CLASSES)}

    def line_operator(self):
        return self.lib.lise_line_operator(self._h).decode()

    def launch_count(self):
        return int(self.lib.lise_launch_count(self._h))

    def device_bytes(self):
        return int(self.lib.lise_device_bytes(self._h))


def _on_device(method):
    """run a Lise method with the context's device current (the C library launches on the current device)."""
    import functools

    @functools.wraps(method)
    def wrapper(self, *a, **k):
        with torch.cuda.device(self.device):
            return method(self, *a, **k)
    return wrapper


for _name in ("observables_ext", "boost", "set_external_fields", "close", "set_params", "set_stream", "set_density_group", "set_dt", "set_chunk", "set_overlap",
              "set_wavefunctions", "get_wavefunctions", "upload_wavefunctions", "download_wavefunctions",
              "set_reduce_hook", "densities", "potentials", "apply_h", "step", "observables", "profile", "profile_read"):
    setattr(Lise, _name, _on_device(getattr(Lise, _name)))
