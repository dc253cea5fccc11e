"""ctypes binding of libsws_jfnk (include/sws_jfnk.h): the linear-Jacobian preconditioner
(section 4.2, App. B/C), right-preconditioned GMRES and damped Newton (section 4.1)
around libsws.  Argument marshalling only; every step runs in the library's kernels.  There
is no CPU fallback: without libsws_jfnk.so the import of the library raises."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from . import SWS_ECUDA, SWS_OK, Context, SwsError, SwsParams, load_library

LIB_PATH = Path(__file__).resolve().parent / "libsws_jfnk.so"

SYMBOLS = (
    "sws_precond_create", "sws_precond_apply", "sws_precond_apply_multi", "sws_precond_block_host", "sws_precond_bytes",
    "sws_precond_bandwidth", "sws_precond_setup_ms", "sws_precond_destroy",
    "sws_solver_create", "sws_solver_gmres", "sws_solver_newton", "sws_solver_continuation", "sws_solver_destroy",
    "sws_jfnk_last_error", "sws_solver_last_error",
)


class GmresOpts(C.Structure):
    _fields_ = [("tol", C.c_double), ("restart", C.c_int32), ("maxit", C.c_int32), ("jv_mode", C.c_int32),
                ("block", C.c_int32)]


class GmresStats(C.Structure):
    _fields_ = [("its", C.c_int32), ("converged", C.c_int32), ("rel_res", C.c_double), ("rhs_norm", C.c_double)]


class NewtonOpts(C.Structure):
    _fields_ = [("ftol", C.c_double), ("eta", C.c_double), ("alpha", C.c_double), ("max_newton", C.c_int32),
                ("max_halvings", C.c_int32), ("gmres", GmresOpts), ("forcing", C.c_int32), ("eta_max", C.c_double)]


class NewtonLog(C.Structure):
    _fields_ = [("newton", C.c_int32), ("gmres_its", C.c_int32), ("fnorm", C.c_double), ("finf", C.c_double),
                ("gmres_rel", C.c_double), ("lambda_", C.c_double)]


class NewtonStats(C.Structure):
    _fields_ = [("steps", C.c_int32), ("converged", C.c_int32), ("residual_evals", C.c_int32),
                ("jv_products", C.c_int32), ("precond_applies", C.c_int32), ("ms_total", C.c_double),
                ("ms_jv", C.c_double), ("ms_precond", C.c_double), ("ms_residual", C.c_double)]


_lib = None


def load_jfnk() -> C.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    load_library()  # libsws.so first, RTLD_GLOBAL
    if not LIB_PATH.exists():
        raise SwsError(f"{LIB_PATH} is missing: run `python -m paper_1403_5044_b200.build`. There is no CPU fallback.")
    lib = C.CDLL(str(LIB_PATH))
    vp, dp = C.c_void_p, C.c_void_p
    proto = {
        "sws_precond_create": (C.c_int, [C.POINTER(SwsParams), C.c_int32, C.c_int32, C.POINTER(vp)]),
        "sws_precond_apply": (C.c_int, [vp, dp, dp, vp]),
        "sws_precond_apply_multi": (C.c_int, [vp, dp, C.c_int32, dp, vp]),
        "sws_precond_block_host": (C.c_int, [vp, C.c_int32, C.c_int32, C.c_int32, dp]),
        "sws_precond_bytes": (C.c_size_t, [vp]),
        "sws_precond_bandwidth": (C.c_int, [vp]),
        "sws_precond_setup_ms": (C.c_double, [vp]),
        "sws_precond_destroy": (C.c_int, [vp]),
        "sws_solver_create": (C.c_int, [vp, vp, C.c_int32, C.POINTER(vp)]),
        "sws_solver_gmres": (C.c_int, [vp, dp, dp, C.POINTER(GmresOpts), dp, C.POINTER(GmresStats), dp, vp]),
        "sws_solver_newton": (C.c_int, [vp, dp, C.POINTER(NewtonOpts), C.POINTER(NewtonLog), C.POINTER(C.c_int32),
                                        C.POINTER(NewtonStats), vp]),
        "sws_solver_continuation": (C.c_int, [vp, dp, dp, C.c_int32, C.POINTER(NewtonOpts),
                                              C.POINTER(NewtonStats), C.POINTER(C.c_int32), vp]),
        "sws_solver_destroy": (C.c_int, [vp]),
        "sws_jfnk_last_error": (C.c_char_p, []),
        "sws_solver_last_error": (C.c_char_p, []),
    }
    for name, (res, args) in proto.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _check(rc: int, what: str) -> None:
    if rc != SWS_OK:
        lib, base = load_jfnk(), load_library()
        msg = base.sws_strerror(rc).decode()
        if rc == SWS_ECUDA:
            msg += ": " + (lib.sws_jfnk_last_error().decode() or lib.sws_solver_last_error().decode()
                           or base.sws_last_cuda_error().decode())
        raise SwsError(f"{what} failed ({rc}): {msg}")


def _params_struct(params: dict, device: int) -> SwsParams:
    return SwsParams(int(params["N"]), int(params["M"]), float(params["x1"]), float(params["y1"]),
                     float(params["dx"]), float(params["dy"]), float(params["froude"]), float(params["eps"]),
                     float(params["n_rad"]), int(params.get("dy_scheme", 0)), 0, 0, int(device))


def _stream(stream=None) -> C.c_void_p:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class Preconditioner:
    """sws_precond_create / sws_precond_destroy.  bandwidth: odd block bandwidth b (L241);
    0 keeps the whole dense block D."""

    def __init__(self, params: dict, bandwidth: int = 0, device: int = 0, factorise: bool = True,
                 f32_panels: bool = False):
        self._h = None
        self.lib = load_jfnk()
        self.n1 = int(params["N"]) + 1
        self.n = 2 * self.n1 * int(params["M"])
        self.device = int(device)
        h = C.c_void_p()
        p = _params_struct(params, device)
        flags = (0 if factorise else 1) | (2 if f32_panels else 0)   # bit 1: factor panels stored in FP32
        _check(self.lib.sws_precond_create(C.byref(p), int(bandwidth), flags, C.byref(h)),
               "sws_precond_create")
        self._h = h

    def close(self) -> None:
        if self._h is not None:
            self.lib.sws_precond_destroy(self._h)
            self._h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def apply(self, v, out=None, stream=None):
        """P^-1 v on device tensors (float64, contiguous, length n)."""
        import torch
        assert v.is_cuda and v.dtype == torch.float64 and v.is_contiguous() and v.numel() == self.n
        if out is None:
            out = torch.empty_like(v)
        _check(self.lib.sws_precond_apply(self._h, v.data_ptr(), out.data_ptr(), _stream(stream)), "sws_precond_apply")
        return out

    def apply_multi(self, V, out=None, stream=None):
        """P^-1 v_q for the t rows of V [t, n] in one sweep over the factor panels (sws_precond_apply_multi)."""
        import torch
        assert V.is_cuda and V.dtype == torch.float64 and V.is_contiguous() and V.dim() == 2 and V.shape[1] == self.n
        if out is None:
            out = torch.empty_like(V)
        _check(self.lib.sws_precond_apply_multi(self._h, V.data_ptr(), int(V.shape[0]), out.data_ptr(),
                                                _stream(stream)), "sws_precond_apply_multi")
        return out

    def block(self, which: int, l: int, m: int) -> np.ndarray:
        out = np.empty((self.n1, self.n1))
        _check(self.lib.sws_precond_block_host(self._h, int(which), int(l), int(m), out.ctypes.data_as(C.c_void_p)),
               "sws_precond_block_host")
        return out

    @property
    def bytes(self) -> int:
        return int(self.lib.sws_precond_bytes(self._h))

    @property
    def bandwidth(self) -> int:
        return int(self.lib.sws_precond_bandwidth(self._h))

    @property
    def setup_ms(self) -> float:
        return float(self.lib.sws_precond_setup_ms(self._h))


class Solver:
    """sws_solver_create / sws_solver_destroy for a Context (max_batch >= 1) and an optional
    Preconditioner."""

    def __init__(self, ctx: Context, precond: Preconditioner | None = None, max_restart: int = 50):
        self._h = None
        self.lib = load_jfnk()
        self.ctx, self.pc = ctx, precond
        h = C.c_void_p()
        _check(self.lib.sws_solver_create(ctx._h, precond._h if precond is not None else None, int(max_restart),
                                          C.byref(h)), "sws_solver_create")
        self._h = h
        self.max_restart = int(max_restart)

    def close(self) -> None:
        if self._h is not None:
            self.lib.sws_solver_destroy(self._h)
            self._h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def gmres(self, u, rhs, tol: float, restart: int | None = None, maxit: int = 200, jv_mode: int = 0,
              block: int = 0, stream=None):
        """Solve J(u) d = rhs; returns (d, stats dict, history array).  block = t >= 2: enlarged GMRES with t
        pieces (history then has one entry per block iteration)."""
        import torch
        restart = self.max_restart if restart is None else int(restart)
        o = GmresOpts(float(tol), restart, int(maxit), int(jv_mode), int(block))
        st = GmresStats()
        hist = np.full(int(maxit), np.nan)
        d = torch.empty_like(u)
        _check(self.lib.sws_solver_gmres(self._h, u.data_ptr(), rhs.data_ptr(), C.byref(o), d.data_ptr(),
                                         C.byref(st), hist.ctypes.data_as(C.c_void_p), _stream(stream)),
               "sws_solver_gmres")
        return d, {"its": st.its, "converged": bool(st.converged), "rel_res": st.rel_res,
                   "rhs_norm": st.rhs_norm}, (hist[:st.its] if block < 2 else hist[~np.isnan(hist)])

    def newton(self, u0, ftol: float = 1e-9, eta: float = 1e-3, restart: int | None = None,
               gmres_maxit: int = 200, max_newton: int = 30, alpha: float = 1e-4, max_halvings: int = 20,
               jv_mode: int = 0, forcing: int = 0, eta_max: float = 0.5, block: int = 0, stream=None):
        """Damped Newton from u0 (device tensor, not modified); returns (u, log list, stats dict)."""
        restart = self.max_restart if restart is None else int(restart)
        o = NewtonOpts(float(ftol), float(eta), float(alpha), int(max_newton), int(max_halvings),
                       GmresOpts(float(eta), restart, int(gmres_maxit), int(jv_mode), int(block)), int(forcing),
                       float(eta_max))
        log = (NewtonLog * (int(max_newton) + 1))()
        nlog = C.c_int32(0)
        st = NewtonStats()
        u = u0.clone()
        _check(self.lib.sws_solver_newton(self._h, u.data_ptr(), C.byref(o), log, C.byref(nlog), C.byref(st),
                                          _stream(stream)), "sws_solver_newton")
        entries = [{"newton": e.newton, "fnorm": e.fnorm, "finf": e.finf, "gmres_its": e.gmres_its,
                    "gmres_rel": e.gmres_rel, "lambda": e.lambda_} for e in log[:nlog.value]]
        stats = {f: getattr(st, f) for f, _ in NewtonStats._fields_}
        stats["converged"] = bool(stats["converged"])
        return u, entries, stats

    def continuation(self, u0, eps_values, ftol: float = 1e-9, eta: float = 1e-3, restart: int | None = None,
                     gmres_maxit: int = 200, max_newton: int = 30, alpha: float = 1e-4, max_halvings: int = 20,
                     jv_mode: int = 0, forcing: int = 0, eta_max: float = 0.5, stream=None):
        """The bootstrapping process of PAPER.md L229: Newton for each source strength in `eps_values`, each
        started from the previous solution.  Returns (u, list of stats dicts of the values that were run,
        number of values that converged).  The context keeps the last epsilon."""
        restart = self.max_restart if restart is None else int(restart)
        o = NewtonOpts(float(ftol), float(eta), float(alpha), int(max_newton), int(max_halvings),
                       GmresOpts(float(eta), restart, int(gmres_maxit), int(jv_mode), 0), int(forcing), float(eta_max))
        eps = np.ascontiguousarray(eps_values, dtype=np.float64)
        st = (NewtonStats * eps.size)()
        ndone = C.c_int32(0)
        u = u0.clone()
        _check(self.lib.sws_solver_continuation(self._h, u.data_ptr(), eps.ctypes.data_as(C.c_void_p), int(eps.size),
                                                C.byref(o), st, C.byref(ndone), _stream(stream)),
               "sws_solver_continuation")
        ran = min(eps.size, ndone.value + 1)
        out = []
        for e in st[:ran]:
            d = {f: getattr(e, f) for f, _ in NewtonStats._fields_}
            d["converged"] = bool(d["converged"])
            out.append(d)
        return u, out, int(ndone.value)
