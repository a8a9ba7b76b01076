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


def _lm_sets(torch, V, N, K):
    z = lambda *s: torch.zeros(s)
    one = lambda lead: {"means3D": z(*lead, N, 3), "scales": z(*lead, N, 3), "quats": z(*lead, N, 4),
                        "opacities": z(*lead, N), "sh": z(*lead, N, K, 3)}
    return one((V,)), one(()), one(())


def test_lm_solve_binding_refuses_masks_and_sets_it_would_misread():
    """The kernels read `update` / `view_touched` as int32 [N] / [V,N] and index the parameter sets by N and K from raw
    pointers: a bool or int64 mask, or a set of another N / K, must be refused by the binding (host logic, no GPU: the
    checks come before any pointer is taken)."""
    import torch
    from types import SimpleNamespace
    from paper_2606_15924_b200.binding import TGS
    V, N, D, K = 2, 8, 3, 16
    g, m, v = _lm_sets(torch, V, N, K)
    call = lambda **kw: TGS.lm_solve(SimpleNamespace(), D, g, m, v, want_delta=False, params=m, **kw)
    for bad in (torch.ones(N, dtype=torch.bool), torch.ones(N, dtype=torch.int64), torch.ones(N + 1, dtype=torch.int32)):
        with pytest.raises(ValueError, match="update must be an int32"):
            call(update=bad)
    for bad in (torch.ones((V, N), dtype=torch.bool), torch.ones((N, V), dtype=torch.int32), torch.ones(N, dtype=torch.int32)):
        with pytest.raises(ValueError, match="view_touched must be an int32"):
            call(view_touched=bad)
    _, m9, _ = _lm_sets(torch, V, N, 9)
    with pytest.raises(ValueError, match=r"m\['sh'\] has shape"):
        TGS.lm_solve(SimpleNamespace(), D, g, m9, v, want_delta=False, params=m)
    _, _, v7 = _lm_sets(torch, V, N - 1, K)
    with pytest.raises(ValueError, match=r"v\['means3D'\] has shape"):
        TGS.lm_solve(SimpleNamespace(), D, g, m, v7, want_delta=False, params=m)
    g65, _, _ = _lm_sets(torch, 65, N, K)
    with pytest.raises(ValueError, match="V = 65"):
        TGS.lm_solve(SimpleNamespace(), D, g65, m, v, want_delta=False, params=m)


def test_sparse_iteration_refuses_misaligned_view_slices_at_construction():
    """View i's SH gradients are a slice of one [V,N,K,3] buffer moved with 16-byte accesses: with K = 9 (or 1) and
    N % 4 != 0 the slices of views 1.. are misaligned.  That is an error at construction, with the remedy in words, not a
    TgsError from the first backward of the first iteration."""
    from types import SimpleNamespace
    import paper_2606_15924_b200 as pk
    cam = pk.Camera()
    cam.width, cam.height, cam.fx, cam.fy = 64, 64, 50.0, 50.0
    for D in (2, 0):
        with pytest.raises(ValueError, match="multiple of 4"):
            pk.SparseIteration(SimpleNamespace(device="cpu"), [cam, cam], 1001, D, 1000)
