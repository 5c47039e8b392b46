"""Thin Python binding of the libptflash C ABI (include/ptflash.h): argument marshalling only.

Every numerical step runs in the CUDA kernels behind the ABI.  PyTorch is used for device memory and
streams, nothing else.  There is NO fallback: if libptflash.so is missing or fails to load, every
entry point raises (build it with `python -m paper_2205_03090_b200.build`).
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_HERE = Path(__file__).resolve().parent
_LIB_PATH = _HERE / "libptflash.so"
_lib = None

PTFLASH_OK, PTFLASH_EINVAL, PTFLASH_ECUDA = 0, -1, -2
ST_STAB_CAP, ST_SPLIT_CAP, ST_BAND, ST_SPLIT_FAILED, ST_LNK0_REJECTED = 1, 2, 4, 8, 32
FLAG_SKIP_STABILITY, FLAG_USE_LNK0 = 1, 2
OPTIONS = ["tol_ss", "tol_newton_g", "tol_newton_step", "probe_margin", "trivial_tol", "band", "probe_iters",
           "stab_ss_iters", "stab_tr_iters", "split_ss_iters", "split_tr_iters", "use_newton", "ss_cap", "engine", "stage_profile", "tol_newton_step_stab", "hint_ss_cap", "split_trivial_tol", "stability_only", "host_chunks", "hint_eta_search", "hint_tr_cap", "early_split_ss", "host_row_copies"]
EXPORTS = ["ptflash_create", "ptflash_flash", "ptflash_flash_ex", "ptflash_flash_host", "ptflash_destroy",
           "ptflash_set_option", "ptflash_get_option", "ptflash_get_stats", "ptflash_get_stage_ms", "ptflash_fp64_peak",
           "ptflash_last_error", "ptflash_version", "ptflash_math_probe", "ptflash_rachford_rice", "ptflash_flash_host_async", "ptflash_host_wait",
           "ptflash_flash_static"]
STATIC_MAX_N = 32768   # PTFLASH_STATIC_MAX_N


class PTFlashError(RuntimeError):
    pass


class _Io(C.Structure):
    _fields_ = [("N", C.c_int64), ("z", C.c_void_p), ("P", C.c_void_p), ("T", C.c_void_p), ("lnK0", C.c_void_p),
                ("flags", C.c_void_p), ("out_beta", C.c_void_p), ("out_x", C.c_void_p), ("out_y", C.c_void_p),
                ("out_phase", C.c_void_p), ("out_iters", C.c_void_p), ("out_tpd_min", C.c_void_p),
                ("out_lnK", C.c_void_p), ("out_status", C.c_void_p), ("out_stab_iters", C.c_void_p),
                ("out_dbeta_dK", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = ([(k, C.c_int64) for k in ("n_total", "n_invalid", "n_probe_case1", "n_probe_case2", "n_probe_case3",
                                          "n_stability", "n_stab_newton", "n_split", "n_split_newton", "n_two_phase",
                                          "kernel_launches")]
                + [("n_stab_tr", C.c_int64 * 2), ("n_stab_capped", C.c_int64 * 2), ("n_split_capped", C.c_int64),
                   ("n_warm_restarts", C.c_int64), ("max_probe_iters", C.c_int32), ("max_stab_ss_iters", C.c_int32 * 2),
                   ("max_stab_tr_iters", C.c_int32 * 2), ("max_split_ss_iters", C.c_int32), ("max_split_tr_iters", C.c_int32),
                   ("reserved_", C.c_int32)])

    def as_dict(self):
        d = {}
        for k, _ in self._fields_:
            v = getattr(self, k)
            if k != "reserved_":
                d[k] = int(v) if isinstance(v, int) else [int(e) for e in v]
        return d


def load_library():
    """Load libptflash.so (once).  Raises PTFlashError if it is not built -- there is no CPU path."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise PTFlashError(f"{_LIB_PATH} not found: the CUDA extension is not built "
                           "(run `python -m paper_2205_03090_b200.build`); there is no CPU fallback")
    L = C.CDLL(str(_LIB_PATH))
    vp, dp, i64 = C.c_void_p, C.POINTER(C.c_double), C.c_int64
    L.ptflash_create.restype = vp
    L.ptflash_create.argtypes = [C.c_int, dp, dp, dp, dp]
    L.ptflash_flash.restype = C.c_int
    L.ptflash_flash.argtypes = [vp, i64] + [vp] * 9
    L.ptflash_flash_ex.restype = C.c_int
    L.ptflash_flash_ex.argtypes = [vp, C.POINTER(_Io), vp]
    L.ptflash_flash_host.restype = C.c_int
    L.ptflash_flash_host.argtypes = [vp, i64] + [vp] * 9
    L.ptflash_flash_host_async.restype = C.c_int
    L.ptflash_flash_host_async.argtypes = [vp, i64] + [vp] * 8
    L.ptflash_host_wait.restype = C.c_int
    L.ptflash_host_wait.argtypes = [vp]
    L.ptflash_destroy.restype = C.c_int
    L.ptflash_destroy.argtypes = [vp]
    L.ptflash_set_option.restype = C.c_int
    L.ptflash_set_option.argtypes = [vp, C.c_int, C.c_double]
    L.ptflash_get_option.restype = C.c_int
    L.ptflash_get_option.argtypes = [vp, C.c_int, dp]
    L.ptflash_get_stats.restype = C.c_int
    L.ptflash_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.ptflash_get_stage_ms.restype = C.c_int
    L.ptflash_get_stage_ms.argtypes = [vp, C.POINTER(C.c_float), C.c_int]
    L.ptflash_fp64_peak.restype = C.c_int
    L.ptflash_fp64_peak.argtypes = [C.c_int, dp, dp, vp]
    L.ptflash_math_probe.restype = C.c_int
    L.ptflash_math_probe.argtypes = [C.c_int, i64, vp, vp, vp]
    L.ptflash_rachford_rice.restype = C.c_int
    L.ptflash_rachford_rice.argtypes = [vp, i64] + [vp] * 7
    L.ptflash_flash_static.restype = C.c_int
    L.ptflash_flash_static.argtypes = [C.c_int, dp, dp, dp, dp, i64] + [vp] * 9
    L.ptflash_last_error.restype = C.c_char_p
    L.ptflash_version.restype = C.c_char_p
    _lib = L
    return L


def _check(rc: int, what: str):
    if rc != PTFLASH_OK:
        raise PTFlashError(f"{what} failed ({rc}): {load_library().ptflash_last_error().decode()}")


def _darr(a):
    import numpy as np
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _ptr(t):
    """Device (or host) address of a torch tensor / numpy array; None -> NULL."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous()
        return C.c_void_p(t.data_ptr())
    return C.c_void_p(t.ctypes.data)


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(int(stream))


# ---- the ABI, same names ---------------------------------------------------------------------
def ptflash_create(nc, Tc, Pc, omega, kij=None):
    L = load_library()
    _a, pTc = _darr(Tc)
    _b, pPc = _darr(Pc)
    _c, pom = _darr(omega)
    _d, pk = _darr(kij) if kij is not None else (None, None)
    h = L.ptflash_create(int(nc), pTc, pPc, pom, pk)
    if not h:
        raise PTFlashError("ptflash_create failed: " + L.ptflash_last_error().decode())
    return C.c_void_p(h)


def ptflash_flash(h, N, z, P, T, out_beta, out_x, out_y, out_phase, out_iters=None, stream=None):
    _check(load_library().ptflash_flash(h, int(N), _ptr(z), _ptr(P), _ptr(T), _ptr(out_beta), _ptr(out_x), _ptr(out_y),
                                        _ptr(out_phase), _ptr(out_iters), _stream(stream)), "ptflash_flash")


def ptflash_flash_ex(h, N, z, P, T, out_beta, out_x, out_y, out_phase, out_iters=None, lnK0=None, flags=None,
                     out_tpd_min=None, out_lnK=None, out_status=None, out_stab_iters=None, out_dbeta_dK=None, stream=None):
    io = _Io(int(N), *[(_ptr(t).value if t is not None else None) for t in
                       (z, P, T, lnK0, flags, out_beta, out_x, out_y, out_phase, out_iters, out_tpd_min, out_lnK,
                        out_status, out_stab_iters, out_dbeta_dK)])
    _check(load_library().ptflash_flash_ex(h, C.byref(io), _stream(stream)), "ptflash_flash_ex")


def ptflash_flash_host(h, N, z, P, T, out_beta, out_x, out_y, out_phase, out_iters=None, stream=None):
    _check(load_library().ptflash_flash_host(h, int(N), _ptr(z), _ptr(P), _ptr(T), _ptr(out_beta), _ptr(out_x),
                                             _ptr(out_y), _ptr(out_phase), _ptr(out_iters), _stream(stream)),
           "ptflash_flash_host")


def ptflash_flash_host_async(h, N, z, P, T, out_beta, out_x, out_y, out_phase, out_iters=None):
    _check(load_library().ptflash_flash_host_async(h, int(N), _ptr(z), _ptr(P), _ptr(T), _ptr(out_beta), _ptr(out_x),
                                                   _ptr(out_y), _ptr(out_phase), _ptr(out_iters)), "ptflash_flash_host_async")


def ptflash_host_wait(h):
    _check(load_library().ptflash_host_wait(h), "ptflash_host_wait")


def ptflash_rachford_rice(h, N, lnK, z, out_theta, out_x=None, out_y=None, out_dtheta_dK=None, stream=None):
    _check(load_library().ptflash_rachford_rice(h, int(N), _ptr(lnK), _ptr(z), _ptr(out_theta), _ptr(out_x), _ptr(out_y),
                                                _ptr(out_dtheta_dK), _stream(stream)), "ptflash_rachford_rice")


def ptflash_flash_static(nc, Tc, Pc, omega, kij, N, z, P, T, out_beta, out_x, out_y, out_phase, out_iters=None, stream=None):
    """The flash for callers that must not allocate (a simulator that has given all device memory to its own pool, a
    time-step loop that cannot afford cudaMalloc's device-wide stall, a job on a fixed memory budget): no handle, the
    workspace is a fixed 32 MiB array inside the library, N <= STATIC_MAX_N.  Tc, Pc, omega, kij: host arrays as for
    ptflash_create; the rest as for ptflash_flash, on the current device.  Calls share the workspace: keep them ordered
    on one stream per device.  See include/ptflash.h."""
    L = load_library()
    _a, pTc = _darr(Tc)
    _b, pPc = _darr(Pc)
    _c, pom = _darr(omega)
    _d, pk = _darr(kij) if kij is not None else (None, None)
    _check(L.ptflash_flash_static(int(nc), pTc, pPc, pom, pk, int(N), _ptr(z), _ptr(P), _ptr(T), _ptr(out_beta), _ptr(out_x),
                                  _ptr(out_y), _ptr(out_phase), _ptr(out_iters), _stream(stream)), "ptflash_flash_static")


def ptflash_destroy(h):
    _check(load_library().ptflash_destroy(h), "ptflash_destroy")


def ptflash_set_option(h, key, value):
    k = OPTIONS.index(key) if isinstance(key, str) else int(key)
    _check(load_library().ptflash_set_option(h, k, float(value)), "ptflash_set_option")


def ptflash_get_option(h, key):
    k = OPTIONS.index(key) if isinstance(key, str) else int(key)
    v = C.c_double(0)
    _check(load_library().ptflash_get_option(h, k, C.byref(v)), "ptflash_get_option")
    return v.value


def ptflash_get_stats(h) -> dict:
    s = Stats()
    _check(load_library().ptflash_get_stats(h, C.byref(s)), "ptflash_get_stats")
    return s.as_dict()


STAGE_NAMES = ["init", "probe", "stab_ss", "stab_newton", "stab_decide", "split_ss", "split_newton"]


def ptflash_get_stage_ms(h) -> list:
    """Stage times (ms) of the last call made with the stage_profile option on; [] if it was off."""
    buf = (C.c_float * 24)()
    n = load_library().ptflash_get_stage_ms(h, buf, 24)
    if n < 0:
        _check(n, "ptflash_get_stage_ms")
    return [float(buf[i]) for i in range(n)]


def ptflash_fp64_peak(iters=4096, stream=None):
    """Measured FP64 FLOP/s of an independent-DFMA kernel on the current device -> (flops_per_s, ms)."""
    f, ms = C.c_double(0), C.c_double(0)
    _check(load_library().ptflash_fp64_peak(int(iters), C.byref(f), C.byref(ms), _stream(stream)), "ptflash_fp64_peak")
    return f.value, ms.value


MATH_FN = ["exp_fast", "exp_tab", "log_fast", "log1p_fast", "rcp_fast", "rsqrt_fast", "sqrt_fast", "div_fast_1", "rcp_nr1"]


def ptflash_math_probe(fn, n, x, y, stream=None):
    """y[i] = fn(x[i]) with one of the library's lean fp64 math routines (device arrays); fn: index or name in MATH_FN."""
    k = MATH_FN.index(fn) if isinstance(fn, str) else int(fn)
    _check(load_library().ptflash_math_probe(k, int(n), _ptr(x), _ptr(y), _stream(stream)), "ptflash_math_probe")


def ptflash_version() -> str:
    return load_library().ptflash_version().decode()


# ---- convenience wrapper (allocation only) ----------------------------------------------------
class PTFlash:
    """Owns a handle for one component system; `flash` allocates the outputs with torch and calls the ABI."""

    def __init__(self, Tc, Pc, omega, kij=None, **options):
        self.nc = len(Tc)
        self.h = ptflash_create(self.nc, Tc, Pc, omega, kij)
        for k, v in options.items():
            ptflash_set_option(self.h, k, v)

    @classmethod
    def from_system(cls, system, **options):
        return cls(system.Tc, system.Pc, system.omega, system.kij, **options)

    def set_option(self, key, value):
        ptflash_set_option(self.h, key, value)

    def stats(self):
        return ptflash_get_stats(self.h)

    def stage_ms(self):
        return ptflash_get_stage_ms(self.h)

    def rachford_rice(self, lnK, z, stream=None):
        """lnK, z [nc, N] CUDA float64 -> dict(theta [N], x, y, dtheta_dK [nc, N])."""
        import torch
        assert z.is_cuda and z.dtype == torch.float64 and z.shape[0] == self.nc and lnK.shape == z.shape
        N = z.shape[1]
        f64 = dict(dtype=torch.float64, device=z.device)
        out = dict(theta=torch.empty(N, **f64), x=torch.empty(self.nc, N, **f64), y=torch.empty(self.nc, N, **f64),
                   dtheta_dK=torch.empty(self.nc, N, **f64))
        ptflash_rachford_rice(self.h, N, lnK, z, out["theta"], out["x"], out["y"], out["dtheta_dK"], stream=stream)
        return out

    def flash(self, z, P, T, lnK0=None, flags=None, extended=True, stream=None):
        """z [nc, N], P [N], T [N]: CUDA float64 tensors -> dict of CUDA tensors."""
        import torch
        assert z.is_cuda and z.dtype == torch.float64 and z.shape[0] == self.nc
        N = z.shape[1]
        dev = z.device
        f64 = dict(dtype=torch.float64, device=dev)
        i32 = dict(dtype=torch.int32, device=dev)
        out = dict(beta=torch.empty(N, **f64), x=torch.empty(self.nc, N, **f64), y=torch.empty(self.nc, N, **f64),
                   phase=torch.empty(N, **i32), iters=torch.empty(N, **i32))
        if extended:
            out.update(tpd_min=torch.empty(N, **f64), lnK=torch.empty(self.nc, N, **f64),
                       status=torch.empty(N, **i32), stab_iters=torch.empty(N, **i32), dbeta_dK=torch.empty(self.nc, N, **f64))
            ptflash_flash_ex(self.h, N, z, P, T, out["beta"], out["x"], out["y"], out["phase"], out["iters"],
                             lnK0=lnK0, flags=flags, out_tpd_min=out["tpd_min"], out_lnK=out["lnK"],
                             out_status=out["status"], out_stab_iters=out["stab_iters"], out_dbeta_dK=out["dbeta_dK"],
                             stream=stream)
        else:
            ptflash_flash(self.h, N, z, P, T, out["beta"], out["x"], out["y"], out["phase"], out["iters"], stream=stream)
        return out

    def close(self):
        if self.h is not None:
            ptflash_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
