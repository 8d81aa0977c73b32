"""CPU-side checks of the boundary: the library builds for sm_100a, loads without a GPU, exports every symbol
include/gcoreccd.h declares, and the Python struct mirrors the C struct."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2203_11043_b200 import build
    return build.build()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "gcoreccd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gcoreccd_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for need in ("gcoreccd_create", "gcoreccd_load_carriers", "gcoreccd_step", "gcoreccd_run_to_collection",
                 "gcoreccd_read_image"):
        assert need in names


def test_library_exports_every_declared_symbol(libpath):
    L = C.CDLL(libpath)
    for name in _declared_symbols():
        assert hasattr(L, name), name
    from paper_2203_11043_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_symbols()


def test_library_is_sm100a_only_and_uses_packed_fp32(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out and "sm_80" not in out
    sass = subprocess.run(["cuobjdump", "-sass", libpath], capture_output=True, text=True).stdout
    for op in ("FFMA2", "FADD2", "FMUL2", "MUFU.RSQ"):
        assert op in sass, op


def test_no_compute_entry_points_work_without_gpu(libpath):
    from paper_2203_11043_b200 import binding
    L = binding.lib()
    assert binding.version().startswith("gcoreccd-b200")
    assert binding.strerror(0) == "ok" and "capacity" in binding.strerror(-3)
    assert binding.workspace_size(0, 64, 64) == 0 and binding.workspace_size(1024, 0, 64) == 0
    n1, n2 = binding.workspace_size(1024, 64, 64), binding.workspace_size(1 << 20, 256, 256)
    assert 0 < n1 < n2 and n1 % 256 == 0
    # create must fail (not fall back) when there is no sm_100 device / bad params
    p = binding.Params()
    h = C.c_void_p()
    assert L.gcoreccd_create(C.byref(p), C.byref(h)) == binding.ERR_INVALID       # struct_size = 0
    assert L.gcoreccd_create(None, C.byref(h)) == binding.ERR_INVALID
    import torch
    if not torch.cuda.is_available():
        p = binding.Params(C.sizeof(binding.Params), 0, 140.0, 2.81e4, 2e3, 675.0, 0.0, 15.0, 0.05, 1e-3, 11.7, 1,
                           64, 64, -480.0, -480.0, -1, 0, None, None, 0, 1024)
        assert L.gcoreccd_create(C.byref(p), C.byref(h)) == binding.ERR_CUDA
        with pytest.raises(RuntimeError):
            binding.Gcoreccd(1024)


def test_params_struct_layout_matches_header():
    from paper_2203_11043_b200 import binding
    # 2 u32 + 9 doubles + u64 + 2 i32 + 2 doubles + 2 i32 + 2 pointers + 2 u64
    assert C.sizeof(binding.Params) == 8 + 72 + 8 + 8 + 16 + 8 + 16 + 16
    assert binding.Params.seed.offset == 80 and binding.Params.stream.offset == 120


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2203_11043_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "goracle" not in txt.replace("oracle/goracle.c", ""), f
    assert "goracle" not in open(os.path.join(ROOT, "include", "gcoreccd.h")).read()
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2203" not in txt and "from paper_2203" not in txt and "gcoreccd.h" not in txt
