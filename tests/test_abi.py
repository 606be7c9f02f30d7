"""CPU-side checks of the boundary: the CUDA library builds, loads, and exports every symbol that
include/lpf.h declares; the ctypes mirrors match the C structs.  No compute calls (no GPU here)."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lpf.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2103_15418_b200 import build, binding
    build.build()
    return binding.load_library()


def binding_w_capacity():
    from paper_2103_15418_b200 import binding
    return binding.W_CAPACITY


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lpf_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert len(names) >= 15 and "lpf_cube_qc" in names and "lpf_detect_sources" in names
    assert "lpf_measure_flux" in names and "lpf_append_dynspec" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in lpf.h but not exported"
    from paper_2103_15418_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_struct_layouts_match_header(tmp_path):
    from paper_2103_15418_b200 import binding
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include "lpf.h"\nint main(){printf("%zu %zu %zu %zu\\n", sizeof(lpf_params), '
                   'sizeof(lpf_det), sizeof(lpf_frame_view), sizeof(lpf_host_result));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)])
    a, b, c, d = map(int, subprocess.check_output([str(exe)]).split())
    assert C.sizeof(binding.LpfParams) == a
    assert binding.DET_DTYPE.itemsize == b == 24
    assert C.sizeof(binding.LpfFrameView) == c
    assert C.sizeof(binding.LpfHostResult) == d


def test_version_and_errors_without_gpu(lib):
    assert lib.lpf_version() >= 100
    assert lib.lpf_strerror(0) == b"ok" and b"argument" in lib.lpf_strerror(-1)
    # the positive status of SURVEY 8(b) "Errors": a truncated list is a warning, not an error
    hdr = open(HEADER).read()
    assert re.search(r"#define\s+LPF_W_CAPACITY\s+1\b", hdr) and binding_w_capacity() == 1
    assert b"truncated" in lib.lpf_strerror(1)
    assert "force_general" in hdr and "getenv" not in open(os.path.join(ROOT, "paper_2103_15418_b200", "csrc", "detect_fused.cu")).read()
    # bad parameters are rejected before any CUDA call
    from paper_2103_15418_b200 import binding, synth
    p = synth.default_params(1); p["B"] = 0
    h = C.c_void_p()
    assert lib.lpf_create(C.byref(h), C.byref(binding.make_params(p)), None) == -1
    import torch
    if not torch.cuda.is_available():
        # no device: the product path fails loudly, it never falls back to the CPU
        p = synth.default_params(1)
        assert lib.lpf_create(C.byref(h), C.byref(binding.make_params(p)), None) == -2
        with pytest.raises(binding.LpfError):
            binding.LPF(p)


def test_product_does_not_touch_the_oracle():
    # the CUDA package and bench's product arm never import oracle/ (parity would be void otherwise)
    pkg = os.path.join(ROOT, "paper_2103_15418_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "lpf_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "lpf_oracle.cpp")).read()
    assert "paper_2103_15418_b200" not in otxt.replace("``paper_2103_15418_b200``", "").replace("(paper_2103_15418_b200/csrc)", "")
