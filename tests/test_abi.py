"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol the
header declares; argument validation that needs no device; loud failure without a device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1909_05423_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def header_functions():
    src = open(os.path.join(ROOT, "include", "pittpack_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pp_[a-z_]+)\s*\(", src)))


def test_header_declares_the_expected_entry_points():
    names = header_functions()
    for must in ("pp_plan_create", "pp_solve", "pp_plan_destroy", "pp_plan_workspace_bytes", "pp_strerror"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in header_functions():
        assert hasattr(lib, name), name


def test_binding_covers_every_declared_symbol():
    from paper_1909_05423_b200 import binding
    assert sorted(binding.EXPORTS) == header_functions()


def test_signatures_use_no_torch_types():
    src = open(os.path.join(ROOT, "include", "pittpack_b200.h")).read()
    assert "torch" not in src and "at::" not in src and "#include <cuda" not in src


def test_validation_without_device():
    import paper_1909_05423_b200 as pp
    assert pp.pp_plan_create(0, 32, 32, 0.1, 0.1, 0.1, 0, 0, 0)[0] == 1       # non-positive size
    assert pp.pp_plan_create(32, 32, 32, -0.1, 0.1, 0.1, 0, 0, 0)[0] == 1     # non-positive spacing
    assert pp.pp_plan_create(32, 32, 32, 0.1, 0.1, float("nan"), 0, 0, 0)[0] == 1
    assert pp.pp_plan_create(32, 32, 32, 0.1, 0.1, 0.1, 0, 3, 0)[0] == 1      # unknown BC
    assert pp.pp_plan_create(36, 32, 32, 0.1, 0.1, 0.1, 0, 0, 0)[0] == 2      # not 2^k, 3*2^k (k >= 4) or 5*2^k (k >= 4)
    assert pp.pp_plan_create(32, 24, 32, 0.1, 0.1, 0.1, 0, 0, 0)[0] == 2      # 3*2^3: too short for the mixed-radix schedule
    assert pp.pp_plan_create(32, 112, 32, 0.1, 0.1, 0.1, 0, 0, 0)[0] == 2     # 7*2^4
    assert pp.pp_plan_create(32, 4096, 32, 0.1, 0.1, 0.1, 0, 0, 0)[0] == 2    # too long
    assert pp.pp_plan_create(32, 32, 1, 0.1, 0.1, 0.1, 0, 0, 0)[0] == 2       # nz < 2
    assert pp.pp_plan_create(32, 32, 16384 + 1, 0.1, 0.1, 0.1, 0, 0, 0)[0] == 2   # lines up to 16384 rows
    assert pp.pp_plan_create(32, 32, 32768, 0.1, 0.1, 0.1, 0, 0, 1)[0] == 2
    assert pp.binding.pp_plan_set_z_algorithm(0, 1) == 5                      # NULL plan
    assert pp.binding.pp_plan_set_xy_fusion(0, 1) == 5
    assert pp.binding.pp_plan_launches_per_solve(0) == 0
    assert pp.pp_plan_destroy(0) == 0
    assert pp.pp_solve(0, 0, 0) == 5
    assert pp.pp_plan_workspace_bytes(0) == 0
    assert "unknown" in pp.strerror(99)
    assert "sm_100a" in pp.version()


def test_fails_loudly_without_a_device():
    """No CPU fallback: on a box without a GPU plan creation reports PP_ERR_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    import paper_1909_05423_b200 as pp
    st, h = pp.pp_plan_create(32, 32, 32, 0.1, 0.1, 0.1, 0, 0, 2)
    assert st == 4 and h == 0
    with pytest.raises(pp.PittPackError):
        pp.Plan(32, 32, 32, 0.1, 0.1, 0.1, "PPD")


def test_product_path_does_not_import_the_oracle():
    """The product path may not import, call, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1909_05423_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle\b|oracle[/.]poisson|oracle[/.]makhoul|#include\s+\"[^\"]*oracle", re.M)
    for dirpath, _, files in os.walk(pkg):
        for name in files:
            if name.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, name)).read()
                assert not pat.search(text), name


def test_size_rules_host_side():
    """pp_size_supported needs no device: 2^k in [4, 2048], 3*2^k in [48, 1536], 5*2^k in [80, 1280];
    nz in [2, 16384], any boundary condition in z."""
    import paper_1909_05423_b200 as pp
    ok = pp.binding.pp_size_supported
    good = [4, 8, 512, 2048, 48, 96, 192, 384, 768, 1536, 80, 160, 320, 640, 1280]
    bad = [0, 2, 3, 6, 12, 24, 36, 40, 56, 112, 144, 4096, 3072, 2560, 100, 1000]
    for n in good:
        assert ok(n, 64, 32, 1) and ok(64, n, 32, 2), n
    for n in bad:
        assert not ok(n, 64, 32, 1) and not ok(64, n, 32, 0), n
    assert ok(64, 64, 2, 0) and ok(64, 64, 4096, 0) and not ok(64, 64, 1, 0)
    assert ok(64, 64, 16384, 1) and ok(48, 48, 8192, 2)
    for bcz in (0, 1, 2):                        # every nz in [2, 16384] with every boundary condition in z
        for nz in (2, 3, 100, 4096, 4097, 5000, 8200, 8192 + 32, 16383, 16384):
            assert ok(64, 64, nz, bcz), (nz, bcz)
        assert not ok(64, 64, 16385, bcz) and not ok(64, 64, 32768, bcz)
    assert not ok(64, 64, 64, 7)                 # unknown boundary condition
