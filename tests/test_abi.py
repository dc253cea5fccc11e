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


def declared_functions():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(sws_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(sws):
    lib = sws.load_library()
    names = declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in sws.h but not exported by libsws.so"
    assert sorted(sws.SYMBOLS) == names, "binding's SYMBOLS list and sws.h disagree"


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
    for code in (-1, -2, -3, -4):
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
