"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/tgs.h declares; host-only entry points work; without a GPU the product fails loudly
(no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_15924_b200 import build
    build.build()
    from paper_2606_15924_b200 import binding
    return binding.load_library()


def test_header_symbols_are_exported(lib):
    from paper_2606_15924_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "tgs.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(tgs_[a-z_0-9]+)\s*\(", hdr)))
    assert declared == sorted(binding.SYMBOLS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_host_only_entry_points(lib):
    from paper_2606_15924_b200.binding import Camera
    cam = Camera()
    cam.width, cam.height, cam.fx, cam.fy = 980, 545, 900.0, 900.0
    T = 62 * 35
    assert lib.tgs_sample_num_tiles(C.byref(cam), 30, 100) == (30 * T) // 100 == 651
    assert lib.tgs_sample_num_tiles(C.byref(cam), 0, 100) == 1
    assert lib.tgs_sample_num_tiles(C.byref(cam), 100, 100) == T
    assert lib.tgs_sample_num_tiles(C.byref(cam), 1, 0) == -1
    b = C.c_size_t()
    assert lib.tgs_bin_sort_workspace_bytes(100000, 1000000, T, C.byref(b)) == 0 and b.value > 12 * 1000000
    assert lib.tgs_sample_workspace_bytes(C.byref(cam), C.byref(b)) == 0 and b.value >= T * 36
    assert b"tgs" in lib.tgs_version()


def test_no_gpu_no_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    assert lib.tgs_create(C.byref(h), 0) == 3  # TGS_ERR_CUDA
    import paper_2606_15924_b200 as pk
    with pytest.raises(RuntimeError):
        pk.TGS(0)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_15924_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "tgs_oracle" not in src and "liboracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "tgs_oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2606_15924_b200", osrc, flags=re.M)
    assert "libtgs" not in osrc and "csrc" not in osrc.replace("(paper_2606_15924_b200/csrc)", "")
