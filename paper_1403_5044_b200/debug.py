"""Binding of libsws_debug.so (include/sws_debug.h): unit-test hooks of the all-pairs kernel's device
primitives and the FP64 issue-rate probes.  Not part of the product path; used by tests/ and by bench.py's
measurement helpers only."""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import SWS_ECUDA, SWS_OK, SwsError, _PKG, _np_ptr, load_library

LIB_PATH = _PKG / "libsws_debug.so"
SYMBOLS = ("sws_probe_fp64_peak", "sws_probe_fp64_mix", "sws_debug_rsqrt_host", "sws_debug_rsqrt_lo_host", "sws_debug_s2col_host",
           "sws_debug_last_cuda_error")
_lib = None


def load_debug_library() -> C.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise SwsError(f"{LIB_PATH} is missing: run `python -m paper_1403_5044_b200.build`")
    lib = C.CDLL(str(LIB_PATH))
    dp, ip = C.c_void_p, C.POINTER(C.c_int32)
    proto = {
        "sws_probe_fp64_peak": (C.c_int, [C.c_int32, C.POINTER(C.c_double), ip, C.POINTER(C.c_double)]),
        "sws_probe_fp64_mix": (C.c_int, [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
        "sws_debug_rsqrt_host": (C.c_int, [C.c_int32, dp, dp, C.c_int32]),
        "sws_debug_rsqrt_lo_host": (C.c_int, [C.c_int32, dp, C.POINTER(C.c_int32), dp, C.c_int32]),
        "sws_debug_s2col_host": (C.c_int, [C.c_int32, C.c_double, C.c_double, C.c_int32, dp, dp, C.c_int32,
                                           C.c_int32, dp, dp]),
        "sws_debug_last_cuda_error": (C.c_char_p, []),
    }
    for name, (res, args) in proto.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _check(rc: int, what: str) -> None:
    if rc != SWS_OK:
        msg = load_library().sws_strerror(rc).decode()
        if rc == SWS_ECUDA:
            msg += ": " + load_debug_library().sws_debug_last_cuda_error().decode()
        raise SwsError(f"{what} failed ({rc}): {msg}")


def probe_fp64_peak(device: int = 0) -> dict:
    """Register-only DFMA microbenchmark: {'tflops', 'sm_count', 'sm_mhz'} (sws_probe_fp64_peak)."""
    lib = load_debug_library()
    tf, sms, mhz = C.c_double(), C.c_int32(), C.c_double()
    _check(lib.sws_probe_fp64_peak(int(device), C.byref(tf), C.byref(sms), C.byref(mhz)),
           "sws_probe_fp64_peak")
    return dict(tflops=tf.value, sm_count=int(sms.value), sm_mhz=mhz.value)


FP64_MIX_KINDS = ("dfma_2reg", "dfma_3reg", "dadd", "dmul", "dfma11_dadd_dmul_mufu_rsq64h", "dfma11_int3",
                  "dfma_2reg_plus_uniform", "dfma12_mufu_rsq64h_x2", "dfma12_mufu_rsq_f32_x2", "dfma12_ffma_x2",
                  "dfma12_lop3_x2")


def probe_fp64_mix(kind: int, warps_per_sm: int = 16, device: int = 0) -> dict:
    """sws_probe_fp64_mix: FP64 thread-instructions per SM per clock of one instruction mix."""
    lib = load_debug_library()
    r, mhz = C.c_double(), C.c_double()
    _check(lib.sws_probe_fp64_mix(int(device), int(kind), int(warps_per_sm), C.byref(r), C.byref(mhz)),
           "sws_probe_fp64_mix")
    return {"kind": FP64_MIX_KINDS[kind], "warps_per_sm": int(warps_per_sm), "fp64_instr_per_sm_clk": r.value,
            "sm_mhz": mhz.value}


def debug_rsqrt(x: np.ndarray, device: int = 0) -> np.ndarray:
    """The library's device reciprocal square root applied to host values (unit test hook)."""
    lib = load_debug_library()
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty_like(x)
    _check(lib.sws_debug_rsqrt_host(int(device), _np_ptr(x), _np_ptr(y), int(x.size)), "sws_debug_rsqrt_host")
    return y


def debug_rsqrt_lo(x: np.ndarray, lo: np.ndarray, device: int = 0) -> np.ndarray:
    """rsqrt_fp64_lo: the reciprocal square root whose seed carries the caller's low word (unit test hook)."""
    lib = load_debug_library()
    x = np.ascontiguousarray(x, dtype=np.float64)
    lo = np.ascontiguousarray(lo, dtype=np.int32)
    assert lo.shape == x.shape
    y = np.empty_like(x)
    _check(lib.sws_debug_rsqrt_lo_host(int(device), _np_ptr(x), lo.ctypes.data_as(C.POINTER(C.c_int32)), _np_ptr(y),
                                       int(x.size)), "sws_debug_rsqrt_lo_host")
    return y


def debug_s2col(y1: float, dy: float, M: int, c: np.ndarray, g: np.ndarray, device: int = 0, nsums: int = 1):
    """(direct, em): the S2 column sum(s) term by term on the device and by the library's far-field
    expansion (unit test hook, sws_debug_s2col_host).  nsums = 3: arrays [n][3] of the sums of the
    analytic Jacobian action."""
    lib = load_debug_library()
    c = np.ascontiguousarray(c, dtype=np.float64)
    g = np.ascontiguousarray(g, dtype=np.float64)
    shape = (c.size,) if nsums == 1 else (c.size, 3)
    d, e = np.empty(shape), np.empty(shape)
    _check(lib.sws_debug_s2col_host(int(device), float(y1), float(dy), int(M), _np_ptr(c), _np_ptr(g),
                                    int(c.size), int(nsums), _np_ptr(d), _np_ptr(e)), "sws_debug_s2col_host")
    return d, e
