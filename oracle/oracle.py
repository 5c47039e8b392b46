"""ctypes binding + build helper for the CPU oracle (oracle/ptflash_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the CUDA
package (paper_2205_03090_b200) and the CUDA package imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ptflash_oracle.cpp"
_LIBS = {"double": _HERE / "libptflash_oracle.so", "long double": _HERE / "libptflash_oracle_ld.so"}

OPT_NAMES = ["tol_ss", "tol_newton_g", "tol_newton_step", "probe_margin", "trivial_tol", "band",
             "probe_iters", "stab_ss_iters", "stab_tr_iters", "split_ss_iters", "split_tr_iters",
             "use_newton", "ss_cap", "hint_ss_cap", "eta_growth", "eta_ratio", "split_trivial_tol", "stability_only", "hint_tr_cap"]


def build(real: str = "double", force: bool = False) -> Path:
    """Compile the oracle with g++ -O2 (OpenMP only parallelises the batch driver over mixtures)."""
    out = _LIBS[real]
    if not force and out.exists() and out.stat().st_mtime >= _SRC.stat().st_mtime:
        return out
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           f'-DORACLE_REAL={real}', str(_SRC), "-o", str(out)]
    subprocess.run(cmd, check=True)
    return out


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """One component system (Tc, Pc, omega, kij) bound to the oracle library."""

    def __init__(self, Tc, Pc, omega, kij=None, real: str = "double"):
        self.lib = C.CDLL(str(build(real)))
        self.nc = len(Tc)
        self.Tc, self.Pc, self.omega = _f64(Tc), _f64(Pc), _f64(omega)
        self.kij = _f64(kij) if kij is not None else np.zeros((self.nc, self.nc))
        L = self.lib
        L.orc_choose_root.restype = C.c_double
        L.orc_gibbs_of_root.restype = C.c_double
        L.orc_rr_f.restype = C.c_double
        for f in (L.orc_choose_root,):
            f.argtypes = [C.c_double, C.c_double]
        L.orc_gibbs_of_root.argtypes = [C.c_double] * 3
        L.orc_cubic_roots.argtypes = [C.c_double, C.c_double, C.POINTER(C.c_double), C.c_int]
        assert L.orc_num_opts() == len(OPT_NAMES)

    @classmethod
    def from_system(cls, system, real: str = "double"):
        return cls(system.Tc, system.Pc, system.omega, system.kij, real=real)

    # ---- options ----
    def default_opts(self) -> dict:
        o = np.zeros(len(OPT_NAMES))
        self.lib.orc_default_opts(_dp(o))
        return dict(zip(OPT_NAMES, o.tolist()))

    def _opts(self, opts):
        if opts is None:
            return None
        d = self.default_opts()
        d.update(opts)
        return _f64([d[k] for k in OPT_NAMES])

    def _sys(self):
        return (C.c_int(self.nc), _dp(self.Tc), _dp(self.Pc), _dp(self.omega), _dp(self.kij))

    # ---- scalar pieces (for pins) ----
    def cubic_roots(self, A, B, closed=False):
        r = np.zeros(3)
        n = self.lib.orc_cubic_roots(float(A), float(B), _dp(r), 1 if closed else 0)
        return r[:n].copy() if n == 3 else r[:1].copy()

    def choose_root(self, A, B):
        return self.lib.orc_choose_root(float(A), float(B))

    def gibbs_of_root(self, Z, A, B):
        return self.lib.orc_gibbs_of_root(float(Z), float(A), float(B))

    def setup(self, P, T):
        nc = self.nc
        Ai, Bi, Aij = np.zeros(nc), np.zeros(nc), np.zeros((nc, nc))
        self.lib.orc_setup(*self._sys(), C.c_double(P), C.c_double(T), _dp(Ai), _dp(Bi), _dp(Aij))
        return Ai, Bi, Aij

    def lnphi(self, P, T, c, deriv=False):
        nc = self.nc
        c = _f64(c)
        out, Z = np.zeros(nc), C.c_double(0)
        M = np.zeros((nc, nc)) if deriv else None
        self.lib.orc_lnphi(*self._sys(), C.c_double(P), C.c_double(T), _dp(c), _dp(out), C.byref(Z), _dp(M))
        return (out, Z.value, M) if deriv else (out, Z.value)

    def lnphi_many(self, P, T, c):
        """c [n, nc] -> (lnphi [n, nc], Z [n]) at one (P, T)."""
        c = _f64(c)
        n, nc = c.shape
        out, Z = np.zeros((n, nc)), np.zeros(n)
        self.lib.orc_lnphi_many(*self._sys(), C.c_double(P), C.c_double(T), C.c_int64(n), _dp(c), _dp(out), _dp(Z))
        return out, Z

    def wilson(self, P, T):
        out = np.zeros(self.nc)
        self.lib.orc_wilson(C.c_int(self.nc), _dp(self.Tc), _dp(self.Pc), _dp(self.omega),
                            C.c_double(P), C.c_double(T), _dp(out))
        return out

    def rachford_rice(self, K, z):
        K, z = _f64(K), _f64(z)
        th = C.c_double(0)
        ok = self.lib.orc_rachford_rice(C.c_int(len(K)), _dp(K), _dp(z), C.byref(th))
        return (th.value if ok else None)

    def rr_dtheta_dK(self, K, z, theta):
        """Eq. 13: d theta / d K_i at a root (theta, K) of the Rachford-Rice equation."""
        K, z = _f64(K), _f64(z)
        out = np.zeros(len(K))
        self.lib.orc_rr_dtheta_dK(C.c_int(len(K)), _dp(K), _dp(z), C.c_double(theta), _dp(out))
        return out

    def rr_batch(self, lnK, z):
        """lnK, z [nc, N] -> dict(theta [N], x, y, dtheta_dK [nc, N], ok [N]); no window -> NaN, ok = 0."""
        lnK, z = _f64(lnK), _f64(z)
        nc, N = z.shape
        out = dict(theta=np.empty(N), x=np.empty((nc, N)), y=np.empty((nc, N)), dtheta_dK=np.empty((nc, N)),
                   ok=np.empty(N, dtype=np.int32))
        self.lib.orc_rr_batch(C.c_int(nc), C.c_int64(N), _dp(lnK), _dp(z), _dp(out["theta"]), _dp(out["x"]), _dp(out["y"]),
                              _dp(out["dtheta_dK"]), out["ok"].ctypes.data_as(C.POINTER(C.c_int32)))
        return out

    def rr_f(self, K, z, theta):
        K, z = _f64(K), _f64(z)
        return self.lib.orc_rr_f(C.c_int(len(K)), _dp(K), _dp(z), C.c_double(theta))

    def stability_trial(self, P, T, z, lnK, side, opts=None):
        z, lnK = _f64(z), _f64(lnK)
        lnW, res = np.zeros(self.nc), np.zeros(6)
        self.lib.orc_stability_trial(*self._sys(), C.c_double(P), C.c_double(T), _dp(z), _dp(lnK), C.c_int(side),
                                     _dp(self._opts(opts)), _dp(lnW), _dp(res))
        return dict(lnW=lnW, tm=res[0], tpd=res[1], trivial=bool(res[2]), ss_iters=int(res[3]),
                    tr_iters=int(res[4]), capped=bool(res[5]))

    def phase_split(self, P, T, z, lnK, opts=None):
        z, lnK = _f64(z), _f64(lnK)
        nc = self.nc
        x, y, lk, res = np.zeros(nc), np.zeros(nc), np.zeros(nc), np.zeros(7)
        self.lib.orc_phase_split(*self._sys(), C.c_double(P), C.c_double(T), _dp(z), _dp(lnK), _dp(self._opts(opts)),
                                 _dp(x), _dp(y), _dp(lk), _dp(res))
        return dict(theta=res[0], two_phase=bool(res[1]), ss_iters=int(res[2]), tr_iters=int(res[3]),
                    status=int(res[4]), rate=res[5], dc=res[6], x=x, y=y, lnK=lk)

    # ---- the batched flash ----
    def flash(self, z, P, T, lnK0=None, flags=None, opts=None, nthreads: int = 0):
        """z [nc, N], P [N], T [N] -> dict of numpy arrays (same layout as the C ABI of the CUDA library)."""
        z, P, T = _f64(z), _f64(P), _f64(T)
        nc, N = z.shape
        assert nc == self.nc and P.shape == (N,) and T.shape == (N,)
        if nthreads <= 0:
            nthreads = os.cpu_count() or 1
        out = dict(
            beta=np.empty(N), x=np.empty((nc, N)), y=np.empty((nc, N)),
            phase=np.empty(N, dtype=np.int32), iters=np.empty(N, dtype=np.int32),
            tpd_min=np.empty(N), lnK=np.empty((nc, N)), status=np.empty(N, dtype=np.int32),
            stab_iters=np.empty(N, dtype=np.int32), probe_case=np.empty(N, dtype=np.int32),
            diag=np.empty((3, N)), stage=np.empty((13, N), dtype=np.int32), dbeta_dK=np.empty((nc, N)),
        )
        l0 = _f64(lnK0) if lnK0 is not None else None
        fl = np.ascontiguousarray(flags, dtype=np.uint8) if flags is not None else None
        ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32))
        used = self.lib.orc_flash_batch(
            *self._sys(), C.c_int64(N), _dp(z), _dp(P), _dp(T), _dp(l0),
            fl.ctypes.data_as(C.POINTER(C.c_uint8)) if fl is not None else None, _dp(self._opts(opts)),
            _dp(out["beta"]), _dp(out["x"]), _dp(out["y"]), ip(out["phase"]), ip(out["iters"]),
            _dp(out["tpd_min"]), _dp(out["lnK"]), ip(out["status"]), ip(out["stab_iters"]),
            ip(out["probe_case"]), _dp(out["diag"]), ip(out["stage"]), _dp(out["dbeta_dK"]), C.c_int(nthreads))
        out["threads"] = used
        return out


if __name__ == "__main__":
    print(build("double", force=True))
    print(build("long double", force=True))
