"""Build libsws.so, libsws_jfnk.so, libsws_tuning.so and libsws_debug.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1403_5044_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIB = PKG / "libsws.so"
LIB_JFNK = PKG / "libsws_jfnk.so"  # the Newton-Krylov driver: calls libsws through its C-ABI, + cuBLAS/cuSOLVER
SOURCES_JFNK = ["jfnk_precond.cu", "jfnk_solver.cu"]
CUDA_LIB64 = "/usr/local/cuda/lib64"
SOURCES = ["sws_api.cu", "sws_fields.cu", "sws_allpairs.cu", "sws_allpairs_c0.cu", "sws_allpairs_c1.cu",
           "sws_allpairs_f32.cu", "sws_jv_exact.cu", "sws_noalloc.cu"]
# timing / profiling / launch-shape calls (include/sws_tuning.h): links against libsws.so, not part of the boundary
LIB_TUNING = PKG / "libsws_tuning.so"
SOURCES_TUNING = ["sws_tuning.cu"]
# test hooks and FP64 issue-rate probes (include/sws_debug.h): a library of its own, not part of the product
LIB_DEBUG = PKG / "libsws_debug.so"
SOURCES_DEBUG = ["sws_debug.cu", "sws_probe.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found: libsws.so cannot be built (there is no CPU fallback)")


STAMP = PKG / ".build_flags"  # the SWS_NVCC_EXTRA string the three libraries were built with


def _extra() -> list[str]:
    # SWS_NVCC_EXTRA: extra flags for the build-time experiments of DESIGN.md section 6 (e.g. -DSWS_RSQRT_F32SEED);
    # they go to ALL THREE libraries (the debug hooks compile the same headers as the product kernels)
    return os.environ.get("SWS_NVCC_EXTRA", "").split()


def needs_build() -> bool:
    if not LIB.exists() or not LIB_JFNK.exists() or not LIB_DEBUG.exists() or not LIB_TUNING.exists():
        return True
    if (STAMP.read_text() if STAMP.exists() else "") != " ".join(_extra()):
        return True  # built with other experiment flags: stale
    t = min(LIB.stat().st_mtime, LIB_JFNK.stat().st_mtime, LIB_DEBUG.stat().st_mtime, LIB_TUNING.stat().st_mtime)
    deps = [CSRC / s for s in SOURCES + SOURCES_JFNK + SOURCES_DEBUG + SOURCES_TUNING] + [ROOT / "include" / "sws_debug.h", ROOT / "include" / "sws_tuning.h"] + [CSRC / "sws_internal.cuh", CSRC / "sws_stage.cuh", CSRC / "sws_farfield.cuh", CSRC / "sws_pair.cuh",
                                                         CSRC / "sws_const.cuh", CSRC / "sws_allpairs_const.cuh", CSRC / "sws_closed_form.cuh",
                                                         CSRC / "jfnk_internal.cuh", ROOT / "include" / "sws.h",
                                                         ROOT / "include" / "sws_jfnk.h"]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    extra = _extra()
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, f"-I{ROOT / 'include'}"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [str(CSRC / s) for s in SOURCES] + ["-Xlinker", "-soname=libsws.so", "-o", str(LIB)]
    subprocess.run(cmd, check=True)
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, f"-I{ROOT / 'include'}"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [str(CSRC / s) for s in SOURCES_JFNK] + [f"-L{PKG}", "-l:libsws.so", "-lcublas", "-lcusolver",
                                                    "-Xlinker", "-rpath=$ORIGIN", "-Xlinker", f"-rpath={CUDA_LIB64}",
                                                    "-Xlinker", "-soname=libsws_jfnk.so", "-o", str(LIB_JFNK)]
    subprocess.run(cmd, check=True)
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-DSWS_BUILD_DEBUG_HOOKS", f"-I{ROOT / 'include'}"]
    cmd += [str(CSRC / s) for s in SOURCES_DEBUG] + ["-Xlinker", "-soname=libsws_debug.so", "-o", str(LIB_DEBUG)]
    subprocess.run(cmd, check=True)
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, f"-I{ROOT / 'include'}"]
    cmd += [str(CSRC / s) for s in SOURCES_TUNING] + [f"-L{PKG}", "-l:libsws.so", "-Xlinker", "-rpath=$ORIGIN",
                                                      "-Xlinker", "-soname=libsws_tuning.so", "-o", str(LIB_TUNING)]
    subprocess.run(cmd, check=True)
    STAMP.write_text(" ".join(extra))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
