"""ctypes front-end of the CPU oracle (oracle/sws_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports
nothing from the CUDA package and shares no code with it.

`Oracle(precision="f64")` is the plain double program (the timed CPU baseline);
`Oracle(precision="f80")` is the same source compiled with REAL = long double
(x86 80-bit), the accuracy reference.  `Oracle(precision="c80")` is the same source
compiled with REAL = long double _Complex: `jv_exact` evaluates the residual at
u + i h v and returns Im/h, the exact Jacobian action J(u) v (complex-step derivative).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
# SWS_ORACLE_SRC / SWS_ORACLE_LIBDIR: tests/test_oracle_mutations.py points these at a deliberately
# broken copy of the source (and a scratch directory for its builds) to prove the pins catch it.
_SRC = Path(os.environ.get("SWS_ORACLE_SRC", _HERE / "sws_oracle.c"))
_LIBDIR = Path(os.environ.get("SWS_ORACLE_LIBDIR", _HERE))
_LIBS = {"f64": _LIBDIR / "libsws_oracle_f64.so", "f80": _LIBDIR / "libsws_oracle_f80.so",
         "c80": _LIBDIR / "libsws_oracle_c80.so"}
# c80: the same source with REAL = long double _Complex (complex-step derivative, -DCSTEP);
# -fcx-limited-range = textbook complex multiply/divide (no NaN-recovery library calls)
_DEFS = {"f64": ["-DREAL=double"], "f80": ["-DREAL=long double"], "c80": ["-DCSTEP", "-fcx-limited-range"]}


def build(force: bool = False, only: str | None = None) -> None:
    """Compile the oracle with gcc: -O2 -fopenmp, no fast-math, no FMA contraction.
    only: build just that precision's library (what Oracle(precision) needs)."""
    for suf, lib in _LIBS.items():
        if only is not None and suf != only:
            continue
        if not force and lib.exists() and lib.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               *_DEFS[suf], f"-DSUF={suf}", str(_SRC), "-o", str(lib), "-lm"]
        subprocess.run(cmd, check=True)


class _Params(C.Structure):
    _fields_ = [("N", C.c_int), ("M", C.c_int), ("x1", C.c_double), ("y1", C.c_double),
                ("dx", C.c_double), ("dy", C.c_double), ("froude", C.c_double),
                ("eps", C.c_double), ("n_rad", C.c_double), ("dy_scheme", C.c_int)]


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _d(a):
    return a.ctypes.data_as(_dp)


class Oracle:
    def __init__(self, precision: str = "f64"):
        if precision not in _LIBS:
            raise ValueError(precision)
        build(only=precision)
        self.suf = precision
        self.lib = C.CDLL(str(_LIBS[precision]))
        s = precision
        f = self._f = {}
        for name, res, args in [
            ("residual", C.c_int, [C.POINTER(_Params), _dp, _ip, C.c_int, _dp]),
            ("jv", C.c_int, [C.POINTER(_Params), _dp, _dp, C.c_double, _ip, C.c_int, _dp, _dp]),
            ("sigma", C.c_double, [C.c_int, _dp, _dp]),
            ("fields", C.c_int, [C.POINTER(_Params), _dp, _dp, _dp, _dp, _dp]),
            ("e2_terms", C.c_int, [C.POINTER(_Params), _dp, C.c_int, C.c_int, _dp]),
            ("row_abc", C.c_int, [C.POINTER(_Params), _dp, C.c_int, C.c_int, _dp, _dp]),
            ("pair_kernels", None, [C.c_double] * 11 + [_dp]),
            ("s2_integral", C.c_double, [C.c_double] * 9),
            ("box_integral", C.c_double, [C.c_double] * 7),
            ("weight", C.c_double, [C.POINTER(_Params), C.c_int, C.c_int]),
            ("dy_line", C.c_int, [C.c_int, C.c_double, C.c_int, C.c_int, _dp, _dp]),
            ("sizeof_real", C.c_int, []),
        ] + ([("jv_exact", C.c_int, [C.POINTER(_Params), _dp, _dp, _ip, C.c_int, _dp, _dp])]
             if precision == "c80" else []):
            fn = getattr(self.lib, f"sws_oracle_{name}_{s}")
            fn.restype, fn.argtypes = res, args
            f[name] = fn

    # -- helpers ---------------------------------------------------------
    @staticmethod
    def _params(p: dict) -> _Params:
        return _Params(int(p["N"]), int(p["M"]), float(p["x1"]), float(p["y1"]), float(p["dx"]),
                       float(p["dy"]), float(p["froude"]), float(p["eps"]), float(p["n_rad"]),
                       int(p.get("dy_scheme", 0)))

    @staticmethod
    def _n(p: dict) -> int:
        return 2 * (int(p["N"]) + 1) * int(p["M"])

    @staticmethod
    def _rows(rows):
        if rows is None:
            return None, 0, None
        r = np.ascontiguousarray(rows, dtype=np.int32)
        return r.ctypes.data_as(_ip), int(r.size), r

    @staticmethod
    def set_threads(n: int) -> None:
        os.environ["OMP_NUM_THREADS"] = str(int(n))

    # -- the path ----------------------------------------------------------
    def residual(self, p: dict, u, rows=None) -> np.ndarray:
        """E(u) in App. A order.  rows: flat target indices l*(N-1)+k whose E2 rows to
        compute (others NaN); None = all."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        assert u.size == self._n(p)
        E = np.empty_like(u)
        rp, nr, _keep = self._rows(rows)
        rc = self._f["residual"](C.byref(self._params(p)), _d(u), rp, nr, _d(E))
        if rc:
            raise RuntimeError(f"sws_oracle_residual rc={rc}")
        return E

    def sigma(self, u, v) -> float:
        u = np.ascontiguousarray(u, dtype=np.float64)
        v = np.ascontiguousarray(v, dtype=np.float64)
        return float(self._f["sigma"](int(u.size), _d(u), _d(v)))

    def jv(self, p: dict, u, v, sigma: float, rows=None):
        """(JV, E(u_b)) by eq. (25); u_b = fma(sigma, v, u) in FP64."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        v = np.ascontiguousarray(v, dtype=np.float64)
        JV, Ep = np.empty_like(u), np.empty_like(u)
        rp, nr, _keep = self._rows(rows)
        rc = self._f["jv"](C.byref(self._params(p)), _d(u), _d(v), float(sigma), rp, nr, _d(JV), _d(Ep))
        if rc:
            raise RuntimeError(f"sws_oracle_jv rc={rc}")
        return JV, Ep

    def jv_exact(self, p: dict, u, v, rows=None, want_e0: bool = False):
        """J(u) v by complex-step differentiation of the residual (c80 build only)."""
        if self.suf != "c80":
            raise ValueError("jv_exact needs Oracle('c80')")
        u = np.ascontiguousarray(u, dtype=np.float64)
        v = np.ascontiguousarray(v, dtype=np.float64)
        assert u.size == self._n(p) and v.size == u.size
        JV, E0 = np.empty_like(u), np.empty_like(u)
        rp, nr, _keep = self._rows(rows)
        rc = self._f["jv_exact"](C.byref(self._params(p)), _d(u), _d(v), rp, nr, _d(JV), _d(E0))
        if rc:
            raise RuntimeError(f"sws_oracle_jv_exact rc={rc}")
        return (JV, E0) if want_e0 else JV

    # -- pieces for the pins -------------------------------------------------
    def fields(self, p: dict, u):
        """zeta, phi, zeta_y, phi_y on the nodes, each [M, N]."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        M, N = int(p["M"]), int(p["N"])
        out = [np.empty((M, N)) for _ in range(4)]
        rc = self._f["fields"](C.byref(self._params(p)), _d(u), *[_d(o) for o in out])
        if rc:
            raise RuntimeError(f"sws_oracle_fields rc={rc}")
        return out

    def e2_terms(self, p: dict, u, k: int, l: int) -> np.ndarray:
        """[2pi(phi*-x*), eps/rho*, sum w dpsi K1, sum w zeta_x K2, sum w S2, I, zeta_x*] (0-based k,l)."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        out = np.empty(7)
        rc = self._f["e2_terms"](C.byref(self._params(p)), _d(u), int(k), int(l), _d(out))
        if rc:
            raise RuntimeError(f"sws_oracle_e2_terms rc={rc}")
        return out

    def row_abc(self, p: dict, u, k: int, l: int):
        """(A, B, C, zeta*) of L177 / L162 exactly as the row E2_{k,l} of the residual uses them (0-based k, l)."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        out, zs = np.empty(3), C.c_double()
        rc = self._f["row_abc"](C.byref(self._params(p)), _d(u), int(k), int(l), _d(out), C.byref(zs))
        if rc:
            raise RuntimeError(f"sws_oracle_row_abc rc={rc}")
        return float(out[0]), float(out[1]), float(out[2]), float(zs.value)

    def pair_kernels(self, x, y, zeta, zeta_x, zeta_y, xs, ys, zetas, A, B, C_):
        out = np.empty(3)
        self._f["pair_kernels"](x, y, zeta, zeta_x, zeta_y, xs, ys, zetas, A, B, C_, _d(out))
        return out  # K1, K2, S2

    def s2_integral(self, A, B, C_, xs, ys, xa, xb, ya, yb) -> float:
        return float(self._f["s2_integral"](A, B, C_, xs, ys, xa, xb, ya, yb))

    def box_integral(self, A, B, C_, s1, s2, t1, t2) -> float:
        return float(self._f["box_integral"](A, B, C_, s1, s2, t1, t2))

    def weight(self, p: dict, i: int, j: int) -> float:
        return float(self._f["weight"](C.byref(self._params(p)), int(i), int(j)))

    def dy_line(self, f, h: float, scheme: int = 0, first_is_symmetric: bool = True) -> np.ndarray:
        f = np.ascontiguousarray(f, dtype=np.float64)
        m = np.empty_like(f)
        rc = self._f["dy_line"](int(f.size), float(h), int(scheme), int(bool(first_is_symmetric)), _d(f), _d(m))
        if rc:
            raise RuntimeError(f"sws_oracle_dy_line rc={rc}")
        return m

    def sizeof_real(self) -> int:
        return int(self._f["sizeof_real"]())
