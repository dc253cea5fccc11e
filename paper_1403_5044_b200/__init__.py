"""Thin Python binding of libsws.so (include/sws.h): argument marshalling only.

Every step of the path (section 3: reconstruction, all-pairs quadrature,
Bernoulli/radiation rows, assembly; eq. (25): batched finite-difference Jv) runs in the
CUDA kernels behind the C-ABI.  PyTorch is used for device memory and streams only.  There
is no CPU fallback: importing works without a GPU (so that the symbols can be checked), but
creating a `Context` needs a CUDA device and a built libsws.so.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libsws.so"

SWS_OK, SWS_EINVAL, SWS_ENOMEM, SWS_ECUDA, SWS_EBATCH, SWS_ESTATE = 0, -1, -2, -3, -4, -5

# every symbol include/sws.h declares (the boundary: libsws.so)
SYMBOLS = (
    "sws_setup", "sws_residual", "sws_jv_batch", "sws_residual_host", "sws_jv_batch_host",
    "sws_last_sigma", "sws_num_unknowns", "sws_num_targets", "sws_num_sources",
    "sws_workspace_bytes", "sws_destroy", "sws_strerror", "sws_last_cuda_error",
    "sws_jv_exact_batch", "sws_jv_exact_batch_host",
    "sws_get_params", "sws_linearize", "sws_jv_apply",
    "sws_set_farfield", "sws_set_eps", "sws_get_fields_host",
    "sws_set_const_path",
    "sws_fd_shifts_noalloc", "sws_noalloc_last_error",
)
# every symbol include/sws_tuning.h declares (timing / profiling / launch-shape calls: libsws_tuning.so)
TUNING_SYMBOLS = (
    "sws_last_launch_count", "sws_time_allpairs", "sws_time_residual", "sws_set_fused_fields",
    "sws_time_allpairs_lin", "sws_lin_plan_info", "sws_set_profiling", "sws_profile_read", "sws_set_tuning",
    "sws_set_states_per_cta", "sws_const_plan_info", "sws_farfield_stats", "sws_plan_info",
    "sws_tuning_last_cuda_error",
)
TUNING_LIB_PATH = _PKG / "libsws_tuning.so"

NOALLOC_MAX_B = 64  # SWS_NOALLOC_MAX_B of include/sws.h


class SwsParams(C.Structure):
    """sws_params of include/sws.h."""
    _fields_ = [("N", C.c_int32), ("M", C.c_int32), ("x1", C.c_double), ("y1", C.c_double),
                ("dx", C.c_double), ("dy", C.c_double), ("froude", C.c_double), ("eps", C.c_double),
                ("n_rad", C.c_double), ("dy_scheme", C.c_int32), ("precision", C.c_int32),
                ("max_batch", C.c_int32), ("device", C.c_int32)]


class SwsError(RuntimeError):
    pass


_lib = None


def load_library() -> C.CDLL:
    """dlopen libsws.so and declare the prototypes.  Fails loudly if it was not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise SwsError(f"{LIB_PATH} is missing: run `python -m paper_1403_5044_b200.build` "
                       "(nvcc, sm_100a).  There is no CPU fallback.")
    lib = C.CDLL(str(LIB_PATH), mode=C.RTLD_GLOBAL)  # libsws_jfnk.so resolves sws_* against it
    vp, dp, ip = C.c_void_p, C.c_void_p, C.POINTER(C.c_int32)
    proto = {
        "sws_setup": (C.c_int, [C.POINTER(SwsParams), C.POINTER(vp)]),
        "sws_get_params": (C.c_int, [vp, C.POINTER(SwsParams)]),
        "sws_linearize": (C.c_int, [vp, dp, vp]),
        "sws_jv_apply": (C.c_int, [vp, dp, C.c_int32, dp, vp]),
        "sws_residual": (C.c_int, [vp, dp, dp, vp]),
        "sws_jv_batch": (C.c_int, [vp, dp, dp, C.c_int32, dp, dp, dp, dp, vp]),
        "sws_jv_exact_batch": (C.c_int, [vp, dp, dp, C.c_int32, dp, vp]),
        "sws_jv_exact_batch_host": (C.c_int, [vp, dp, dp, C.c_int32, dp, vp]),
        "sws_residual_host": (C.c_int, [vp, dp, dp, vp]),
        "sws_jv_batch_host": (C.c_int, [vp, dp, dp, C.c_int32, dp, dp, dp, dp, vp]),
        "sws_last_sigma": (C.c_int, [vp, C.c_int32, dp, vp]),
        "sws_num_unknowns": (C.c_size_t, [vp]),
        "sws_num_targets": (C.c_size_t, [vp]),
        "sws_num_sources": (C.c_size_t, [vp]),
        "sws_workspace_bytes": (C.c_size_t, [vp]),
        "sws_destroy": (C.c_int, [vp]),
        "sws_strerror": (C.c_char_p, [C.c_int]),
        "sws_last_cuda_error": (C.c_char_p, []),
        "sws_get_fields_host": (C.c_int, [vp, dp, dp, dp, dp, vp]),
        "sws_set_farfield": (C.c_int, [vp, C.c_double]),
        "sws_set_eps": (C.c_int, [vp, C.c_double]),
        "sws_set_const_path": (C.c_int, [vp, C.c_int32]),
        "sws_fd_shifts_noalloc": (C.c_int, [dp, dp, C.c_int64, C.c_int32, dp, C.c_int32, vp]),
        "sws_noalloc_last_error": (C.c_char_p, []),
    }
    for name, (res, args) in proto.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


_tlib = None


def load_tuning_library() -> C.CDLL:
    """dlopen libsws_tuning.so (include/sws_tuning.h): the timing, profiling and launch-shape calls bench.py
    --experiments and the tests use.  Not needed for the hot path."""
    global _tlib
    if _tlib is not None:
        return _tlib
    load_library()  # libsws_tuning.so resolves the context and the launchers against libsws.so
    if not TUNING_LIB_PATH.exists():
        raise SwsError(f"{TUNING_LIB_PATH} is missing: run `python -m paper_1403_5044_b200.build`")
    lib = C.CDLL(str(TUNING_LIB_PATH))
    vp, dp, ip = C.c_void_p, C.c_void_p, C.POINTER(C.c_int32)
    proto = {
        "sws_time_allpairs_lin": (C.c_int, [vp, C.c_int32, C.POINTER(C.c_float), vp]),
        "sws_lin_plan_info": (C.c_int, [vp, C.c_int32, ip]),
        "sws_last_launch_count": (C.c_int, [vp]),
        "sws_time_allpairs": (C.c_int, [vp, C.c_int32, C.c_int32, C.POINTER(C.c_float), vp]),
        "sws_set_tuning": (C.c_int, [vp, C.c_int32]),
        "sws_plan_info": (C.c_int, [vp, C.c_int32, ip]),
        "sws_set_profiling": (C.c_int, [vp, C.c_int32]),
        "sws_profile_read": (C.c_int, [vp, C.POINTER(C.c_double), ip, C.c_int32]),
        "sws_set_states_per_cta": (C.c_int, [vp, C.c_int32]),
        "sws_const_plan_info": (C.c_int, [vp, C.POINTER(C.c_int32)]),
        "sws_time_residual": (C.c_int, [vp, dp, dp, C.c_int32, C.POINTER(C.c_float), vp]),
        "sws_set_fused_fields": (C.c_int, [vp, C.c_int32]),
        "sws_farfield_stats": (C.c_int, [vp, C.c_int32, C.POINTER(C.c_double), vp]),
        "sws_tuning_last_cuda_error": (C.c_char_p, []),
    }
    for name, (res, args) in proto.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _tlib = lib
    return lib


def _check(rc: int, what: str) -> None:
    if rc != SWS_OK:
        lib = load_library()
        msg = lib.sws_strerror(rc).decode()
        if rc == SWS_ECUDA:
            msg += ": " + lib.sws_last_cuda_error().decode()
            if _tlib is not None and what in TUNING_SYMBOLS:
                msg += _tlib.sws_tuning_last_cuda_error().decode()
        raise SwsError(f"{what} failed ({rc}): {msg}")


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _torch():
    import torch
    return torch


def fd_shifts_noalloc(u, V, out, stream=None):
    """sws_fd_shifts_noalloc: out[r] = 1e-7 (1 + |u|_2) / |V[r]|_2 (eq. (25) L219 shifts; 0 for a zero row), with no
    context and no device allocation anywhere in the call - for programs that cannot cudaMalloc where they need the
    shifts (all device memory already handed to the host application's pool; a loop that cannot take cudaMalloc's
    device-wide stall).  The caller therefore brings the output too: u [n], V [b, n], out [b], contiguous float64
    CUDA tensors on one device, b <= NOALLOC_MAX_B.  The scratch of the reduction is one fixed 33 KB array inside
    libsws.so that all calls on a device share: do not let two calls overlap on the GPU (keep them on one stream or
    order them with an event).  Asynchronous on `stream` (default: torch's current stream).  Returns `out`."""
    torch = _torch()
    lib = load_library()
    for name, t in (("u", u), ("V", V), ("out", out)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and t.device == u.device):
            raise SwsError(f"{name}: need a contiguous float64 CUDA tensor on the device of u")
    if u.dim() != 1 or V.dim() != 2 or V.shape[1] != u.shape[0] or tuple(out.shape) != (V.shape[0],):
        raise SwsError("fd_shifts_noalloc: need u [n], V [b, n], out [b]")
    dev_index = u.device.index if u.device.index is not None else torch.cuda.current_device()
    s = stream if stream is not None else torch.cuda.current_stream(dev_index)
    rc = lib.sws_fd_shifts_noalloc(C.c_void_p(u.data_ptr()), C.c_void_p(V.data_ptr()), int(u.shape[0]),
                                   int(V.shape[0]), C.c_void_p(out.data_ptr()), int(dev_index),
                                   C.c_void_p(s.cuda_stream))
    if rc != SWS_OK:
        raise SwsError(f"sws_fd_shifts_noalloc failed ({rc}): {lib.sws_noalloc_last_error().decode()}")
    return out


class Context:
    """sws_setup / sws_destroy.  `params` is a dict with the keys of sws_params (N, M, x1, y1,
    dx, dy, froude, eps, n_rad[, dy_scheme]) - e.g. workloads.Config.params()."""

    def __init__(self, params: dict, max_batch: int = 0, device: int = 0, precision: int = 0):
        self._h = None
        self.lib = load_library()
        self._tlib = None
        p = SwsParams(int(params["N"]), int(params["M"]), float(params["x1"]), float(params["y1"]),
                      float(params["dx"]), float(params["dy"]), float(params["froude"]),
                      float(params["eps"]), float(params["n_rad"]), int(params.get("dy_scheme", 0)),
                      int(precision), int(max_batch), int(device))
        h = C.c_void_p()
        _check(self.lib.sws_setup(C.byref(p), C.byref(h)), "sws_setup")
        self._h = h
        self.device = int(device)
        self.max_batch = int(max_batch)
        self.n = int(self.lib.sws_num_unknowns(h))
        self.targets = int(self.lib.sws_num_targets(h))
        self.sources = int(self.lib.sws_num_sources(h))
        self._N = int(params["N"])

    # -- lifetime ------------------------------------------------------------------
    def close(self) -> None:
        if self._h is not None:
            self.lib.sws_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- helpers ---------------------------------------------------------------------
    @property
    def tlib(self) -> C.CDLL:
        """libsws_tuning.so, loaded on first use (measurement / tuning methods only)."""
        if self._tlib is None:
            self._tlib = load_tuning_library()
        return self._tlib

    def _stream(self, stream=None) -> C.c_void_p:
        torch = _torch()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        return C.c_void_p(s.cuda_stream)

    def _dev(self, t, shape, name):
        torch = _torch()
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64
                and t.is_contiguous() and t.device.index == self.device):
            raise SwsError(f"{name}: need a contiguous float64 CUDA tensor on device {self.device}")
        if tuple(t.shape) != tuple(shape):
            raise SwsError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
        return C.c_void_p(t.data_ptr())

    def _new(self, *shape):
        torch = _torch()
        return torch.empty(shape, dtype=torch.float64, device=f"cuda:{self.device}")

    # -- the path ----------------------------------------------------------------------
    def residual(self, u, out=None, stream=None):
        """F = E(u) on device tensors (sws_residual); asynchronous on the stream."""
        F = out if out is not None else self._new(self.n)
        _check(self.lib.sws_residual(self._h, self._dev(u, (self.n,), "u"),
                                     self._dev(F, (self.n,), "F"), self._stream(stream)), "sws_residual")
        return F

    def jv_batch(self, u, V, sigma=None, want_fpert: bool = False, want_f0: bool = False, stream=None):
        """JV[b] = (E(u + sigma_b v_b) - E(u)) / sigma_b (sws_jv_batch).  sigma: None (device
        formula 1e-7 (1 + |u|) / |v_b|) or b host floats.  Returns JV or (JV, Fpert, F0)."""
        b = int(V.shape[0])
        JV = self._new(b, self.n)
        Fp = self._new(b, self.n) if want_fpert else None
        F0 = self._new(self.n) if want_f0 else None
        sg = None
        if sigma is not None:
            sg = np.ascontiguousarray(sigma, dtype=np.float64)
            if sg.shape != (b,):
                raise SwsError("sigma: need b values")
        rc = self.lib.sws_jv_batch(
            self._h, self._dev(u, (self.n,), "u"), self._dev(V, (b, self.n), "V"), b,
            _np_ptr(sg) if sg is not None else None, C.c_void_p(JV.data_ptr()),
            C.c_void_p(Fp.data_ptr()) if Fp is not None else None,
            C.c_void_p(F0.data_ptr()) if F0 is not None else None, self._stream(stream))
        _check(rc, "sws_jv_batch")
        if want_fpert or want_f0:
            return JV, Fp, F0
        return JV

    def jv_exact_batch(self, u, V, out=None, stream=None):
        """JV[b] = J(u) v_b, the analytic Jacobian action (sws_jv_exact_batch); asynchronous."""
        b = int(V.shape[0])
        JV = out if out is not None else self._new(b, self.n)
        _check(self.lib.sws_jv_exact_batch(self._h, self._dev(u, (self.n,), "u"),
                                           self._dev(V, (b, self.n), "V"), b,
                                           self._dev(JV, (b, self.n), "JV"), self._stream(stream)),
               "sws_jv_exact_batch")
        return JV

    def linearize(self, u, stream=None) -> None:
        """sws_linearize: form and keep everything of J(u) that depends on u alone."""
        _check(self.lib.sws_linearize(self._h, self._dev(u, (self.n,), "u"), self._stream(stream)), "sws_linearize")

    def jv_apply(self, V, out=None, stream=None):
        """sws_jv_apply: J(u) v_b for the u of the last linearize(); V [b, n] or [n]."""
        single = V.dim() == 1
        V2 = V.reshape(1, -1) if single else V
        b = int(V2.shape[0])
        JV = self._new(b, self.n) if out is None else out.reshape(b, -1)
        _check(self.lib.sws_jv_apply(self._h, self._dev(V2, (b, self.n), "V"), b,
                                     self._dev(JV, (b, self.n), "out"), self._stream(stream)), "sws_jv_apply")
        return JV[0] if single else JV

    def jv_exact_batch_host(self, u: np.ndarray, V: np.ndarray, out=None, stream=None) -> np.ndarray:
        """The same on HOST buffers (sws_jv_exact_batch_host): H2D, compute, D2H, synchronise."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        V = np.ascontiguousarray(V, dtype=np.float64)
        b = int(V.shape[0])
        if u.shape != (self.n,) or V.shape != (b, self.n):
            raise SwsError("u/V: wrong shape")
        JV = out if out is not None else np.empty((b, self.n))
        _check(self.lib.sws_jv_exact_batch_host(self._h, _np_ptr(u), _np_ptr(V), b, _np_ptr(JV),
                                                self._stream(stream)), "sws_jv_exact_batch_host")
        return JV

    def residual_host(self, u: np.ndarray, out: np.ndarray | None = None, stream=None) -> np.ndarray:
        """E(u) on HOST buffers (sws_residual_host): H2D copy, compute, D2H copy, synchronise."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        if u.shape != (self.n,):
            raise SwsError("u: wrong length")
        F = out if out is not None else np.empty(self.n)
        _check(self.lib.sws_residual_host(self._h, _np_ptr(u), _np_ptr(F), self._stream(stream)),
               "sws_residual_host")
        return F

    def jv_batch_host(self, u: np.ndarray, V: np.ndarray, sigma=None, out=None, fpert=None, f0=None,
                      stream=None):
        """Batched Jv on HOST buffers (sws_jv_batch_host).  Returns (JV, Fpert, F0)."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        V = np.ascontiguousarray(V, dtype=np.float64)
        b = int(V.shape[0])
        if u.shape != (self.n,) or V.shape != (b, self.n):
            raise SwsError("u/V: wrong shape")
        JV = out if out is not None else np.empty((b, self.n))
        Fp = fpert if fpert is not None else np.empty((b, self.n))
        F0 = f0 if f0 is not None else np.empty(self.n)
        sg = np.ascontiguousarray(sigma, dtype=np.float64) if sigma is not None else None
        rc = self.lib.sws_jv_batch_host(self._h, _np_ptr(u), _np_ptr(V), b,
                                        _np_ptr(sg) if sg is not None else None, _np_ptr(JV),
                                        _np_ptr(Fp), _np_ptr(F0), self._stream(stream))
        _check(rc, "sws_jv_batch_host")
        return JV, Fp, F0

    def fields_host(self, stream=None):
        """sws_get_fields_host: (zeta, phi, zeta_y, phi_y), each [M, N], of the state the last call evaluated."""
        M, N = self.sources // self._N, self._N
        out = [np.empty((M, N)) for _ in range(4)]
        _check(self.lib.sws_get_fields_host(self._h, *[_np_ptr(o) for o in out], self._stream(stream)),
               "sws_get_fields_host")
        return tuple(out)

    def last_sigma(self, b: int, stream=None) -> np.ndarray:
        out = np.empty(int(b))
        _check(self.lib.sws_last_sigma(self._h, int(b), _np_ptr(out), self._stream(stream)), "sws_last_sigma")
        return out

    # -- measurement / tuning ------------------------------------------------------------
    def time_allpairs(self, states: int = 1, reps: int = 1, stream=None) -> float:
        """ms per launch of the all-pairs kernel alone (CUDA events on the stream)."""
        ms = C.c_float()
        _check(self.tlib.sws_time_allpairs(self._h, int(states), int(reps), C.byref(ms),
                                          self._stream(stream)), "sws_time_allpairs")
        return float(ms.value)

    def time_residual(self, u, F, reps: int = 20, stream=None) -> float:
        """ms per sws_residual call, `reps` calls issued back to back inside the library (sws_time_residual)."""
        ms = C.c_float()
        _check(self.tlib.sws_time_residual(self._h, self._dev(u, (self.n,), "u"), self._dev(F, (self.n,), "F"),
                                          int(reps), C.byref(ms), self._stream(stream)), "sws_time_residual")
        return float(ms.value)

    def set_fused_fields(self, on: bool = True) -> None:
        """sws_set_fused_fields: one cooperative launch (default on small meshes) or three for the O(NM) stages."""
        _check(self.tlib.sws_set_fused_fields(self._h, int(bool(on))), "sws_set_fused_fields")

    def time_allpairs_lin(self, reps: int = 1, stream=None) -> float:
        """ms per launch of the analytic-Jv all-pairs kernel alone (after a jv_exact_batch call)."""
        ms = C.c_float()
        _check(self.tlib.sws_time_allpairs_lin(self._h, int(reps), C.byref(ms), self._stream(stream)),
               "sws_time_allpairs_lin")
        return float(ms.value)

    def lin_plan_info(self, b: int) -> dict:
        out = (C.c_int32 * 6)()
        _check(self.tlib.sws_lin_plan_info(self._h, int(b), out), "sws_lin_plan_info")
        return dict(tiles=out[0], chunks=out[1], cols_per_chunk=out[2], seg_len=out[3], nseg=out[4],
                    dirs_per_tile=out[5])

    def set_profiling(self, on: bool = True) -> None:
        _check(self.tlib.sws_set_profiling(self._h, int(bool(on))), "sws_set_profiling")

    def profile_read(self, reset: bool = True):
        """(summed all-pairs kernel ms, launches) since the last reset; synchronises."""
        ms, n = C.c_double(), C.c_int32()
        _check(self.tlib.sws_profile_read(self._h, C.byref(ms), C.byref(n), int(bool(reset))),
               "sws_profile_read")
        return float(ms.value), int(n.value)

    def set_tuning(self, chunks: int = 0) -> None:
        _check(self.tlib.sws_set_tuning(self._h, int(chunks)), "sws_set_tuning")

    def set_states_per_cta(self, ns: int = 0) -> None:
        """sws_set_states_per_cta: states one CTA of a batched all-pairs launch carries (0 default, 1, 2)."""
        _check(self.tlib.sws_set_states_per_cta(self._h, int(ns)), "sws_set_states_per_cta")

    def set_const_path(self, mode: int = -1) -> None:
        """sws_set_const_path: -1 automatic (large meshes), 0 staged kernel only, 1 constant-bank kernel whenever it fits."""
        _check(self.lib.sws_set_const_path(self._h, int(mode)), "sws_set_const_path")

    def const_plan_info(self) -> dict:
        out = (C.c_int32 * 4)()
        _check(self.tlib.sws_const_plan_info(self._h, out), "sws_const_plan_info")
        return dict(active=bool(out[0]), cols_per_slab=out[1], slabs=out[2], tiles=out[3])

    def set_eps(self, eps: float) -> None:
        """sws_set_eps: the source strength of the continuation process."""
        _check(self.lib.sws_set_eps(self._h, float(eps)), "sws_set_eps")

    def set_farfield(self, radius_in_dy: float = 8.0) -> None:
        """sws_set_farfield: <= 0 sums every S2 term directly (the plain definition)."""
        _check(self.lib.sws_set_farfield(self._h, float(radius_in_dy)), "sws_set_farfield")

    def farfield_stats(self, states: int = 1) -> float:
        """Fraction of (warp, column) combinations that take the direct S2 loop."""
        f = C.c_double()
        _check(self.tlib.sws_farfield_stats(self._h, int(states), C.byref(f), self._stream()), "sws_farfield_stats")
        return float(f.value)

    def plan_info(self, states: int = 1) -> dict:
        out = (C.c_int32 * 5)()
        _check(self.tlib.sws_plan_info(self._h, int(states), out), "sws_plan_info")
        return dict(tiles=out[0], chunks=out[1], cols_per_chunk=out[2], seg_len=out[3], nseg=out[4])

    @property
    def last_launch_count(self) -> int:
        return int(self.tlib.sws_last_launch_count(self._h))

    @property
    def workspace_bytes(self) -> int:
        return int(self.lib.sws_workspace_bytes(self._h))
