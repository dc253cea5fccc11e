"""CPU-side checks of the boundary: libsws.so loads without a GPU, exports every symbol
include/sws.h declares, the ctypes mirror of sws_params matches the C layout, and the product
path fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import re
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "sws.h"


@pytest.fixture(scope="module")
def sws():
    import paper_1403_5044_b200 as m
    from paper_1403_5044_b200 import build
    build.build()            # nvcc cross-compiles for sm_100a without a GPU
    m.load_library()
    return m


def declared_functions(header=HEADER):
    text = re.sub(r"/\*.*?\*/", "", header.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(sws_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(sws):
    lib = sws.load_library()
    names = declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in sws.h but not exported by libsws.so"
    assert sorted(sws.SYMBOLS) == names, "binding's SYMBOLS list and sws.h disagree"


def test_tuning_header_symbols_exported(sws):
    """The timing / profiling / launch-shape calls live in libsws_tuning.so (include/sws_tuning.h); the boundary
    library exports none of them and its header declares none of them."""
    lib = sws.load_tuning_library()
    names = declared_functions(ROOT / "include" / "sws_tuning.h")
    assert sorted(names) == sorted(sws.TUNING_SYMBOLS)
    prod = sws.load_library()
    boundary = set(declared_functions())
    for n in names:
        assert hasattr(lib, n), f"{n} declared in sws_tuning.h but not exported by libsws_tuning.so"
        assert not hasattr(prod, n), f"{n} leaked into the product library"
        assert n not in boundary
    assert len(boundary) <= 26, "include/sws.h is the boundary: timing and tuning calls belong in sws_tuning.h"
    assert lib.sws_plan_info(None, 1, None) == sws.SWS_EINVAL and lib.sws_last_launch_count(None) == 0


def test_noalloc_entry_point_validates_before_touching_cuda(sws):
    """sws_fd_shifts_noalloc refuses what its built-in scratch array cannot hold (and bad arguments) with a clear
    message, before any CUDA call: checkable without a GPU."""
    lib = sws.load_library()
    fake = ctypes.c_void_p(256)                                  # never dereferenced: the checks come first
    assert lib.sws_fd_shifts_noalloc(None, fake, 10, 1, fake, 0, None) == sws.SWS_EINVAL
    assert b"NULL" in lib.sws_noalloc_last_error()
    assert lib.sws_fd_shifts_noalloc(fake, fake, 10, sws.NOALLOC_MAX_B + 1, fake, 0, None) == sws.SWS_EBATCH
    assert b"at most 64" in lib.sws_noalloc_last_error()
    assert lib.sws_fd_shifts_noalloc(fake, fake, 10, 0, fake, 0, None) == sws.SWS_EBATCH
    assert lib.sws_fd_shifts_noalloc(fake, fake, 0, 1, fake, 0, None) == sws.SWS_EINVAL
    assert lib.sws_fd_shifts_noalloc(fake, fake, 2 ** 31, 1, fake, 0, None) == sws.SWS_EINVAL
    assert lib.sws_fd_shifts_noalloc(fake, fake, 10, 1, fake, 64, None) == sws.SWS_EINVAL
    text = HEADER.read_text()
    assert "#define SWS_NOALLOC_MAX_B 64" in text and "33,280" in text


def test_debug_header_symbols_exported(sws):
    """libsws_debug.so (test hooks + probes) exports what sws_debug.h declares; the product library has none of them."""
    from paper_1403_5044_b200 import debug
    lib = debug.load_debug_library()
    names = declared_functions(ROOT / "include" / "sws_debug.h")
    assert sorted(names) == sorted(debug.SYMBOLS)
    prod = sws.load_library()
    for n in names:
        assert hasattr(lib, n)
        assert not hasattr(prod, n), f"{n} leaked into the product library"


def test_jfnk_header_symbols_exported(sws):
    """libsws_jfnk.so (Newton-Krylov driver) loads without a GPU and exports what sws_jfnk.h declares."""
    import paper_1403_5044_b200.jfnk as jf
    lib = jf.load_jfnk()
    names = declared_functions(ROOT / "include" / "sws_jfnk.h")
    assert len(names) >= 11
    for n in names:
        assert hasattr(lib, n), f"{n} declared in sws_jfnk.h but not exported by libsws_jfnk.so"
    assert set(names) <= set(jf.SYMBOLS)
    assert lib.sws_precond_create(None, 1, 0, None) == sws.SWS_EINVAL
    assert lib.sws_solver_create(None, None, 10, None) == sws.SWS_EINVAL
    assert lib.sws_precond_destroy(None) == 0 and lib.sws_solver_destroy(None) == 0


def test_jfnk_struct_layouts(sws, tmp_path):
    import paper_1403_5044_b200.jfnk as jf
    structs = {"sws_gmres_opts": jf.GmresOpts, "sws_gmres_stats": jf.GmresStats, "sws_newton_opts": jf.NewtonOpts,
               "sws_newton_log": jf.NewtonLog, "sws_newton_stats": jf.NewtonStats}
    src = tmp_path / "layout2.c"
    body = "".join(f'printf("%zu\\n", sizeof({c}));\n' for c in structs)
    src.write_text('#include <stdio.h>\n#include "sws_jfnk.h"\nint main(void){\n' + body + "return 0;}\n")
    exe = tmp_path / "layout2"
    subprocess.run(["gcc", f"-I{ROOT / 'include'}", str(src), "-o", str(exe)], check=True)
    out = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    for (cname, ct), size in zip(structs.items(), out):
        assert ctypes.sizeof(ct) == size, cname


def test_params_struct_layout(sws, tmp_path):
    """sizeof/offsetof of sws_params as the C compiler sees them == the ctypes mirror."""
    src = tmp_path / "layout.c"
    fields = [f for f, _ in sws.SwsParams._fields_]
    src.write_text(
        '#include <stdio.h>\n#include <stddef.h>\n#include "sws.h"\nint main(void){\n'
        'printf("%zu\\n", sizeof(sws_params));\n'
        + "".join(f'printf("%zu\\n", offsetof(sws_params, {f}));\n' for f in fields)
        + "return 0;}\n")
    exe = tmp_path / "layout"
    subprocess.run(["gcc", f"-I{ROOT / 'include'}", str(src), "-o", str(exe)], check=True)
    out = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    assert out[0] == ctypes.sizeof(sws.SwsParams)
    for f, off in zip(fields, out[1:]):
        assert getattr(sws.SwsParams, f).offset == off, f


def test_error_strings(sws):
    lib = sws.load_library()
    assert lib.sws_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5):
        assert lib.sws_strerror(code) not in (b"ok", b"unknown error")
    assert lib.sws_strerror(-99) == b"unknown error"


def test_null_arguments_rejected(sws):
    lib = sws.load_library()
    assert lib.sws_setup(None, None) == sws.SWS_EINVAL
    assert lib.sws_residual(None, None, None, None) == sws.SWS_EINVAL
    assert lib.sws_destroy(None) == sws.SWS_EINVAL
    assert lib.sws_num_unknowns(None) == 0


def test_no_cpu_fallback(sws):
    """Without a CUDA device the product path must fail, never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import workloads as W
    with pytest.raises(sws.SwsError):
        sws.Context(W.CONFIGS[0].params())


def test_package_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the package imports, includes or loads it."""
    pat = re.compile(r"import\s+oracle|from\s+oracle|#include\s+[\"<].*oracle|sws_oracle|libsws_oracle")
    for f in (ROOT / "paper_1403_5044_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".cuh", ".h"):
            assert not pat.search(f.read_text()), f
    code = ("import sys; import paper_1403_5044_b200, paper_1403_5044_b200.replicas, "
            "paper_1403_5044_b200.build; assert 'oracle' not in sys.modules")
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)
