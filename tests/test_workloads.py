"""The seeded input generators (paper_1909_05423_b200/workloads.py): shapes, spacings, determinism and
the zero-mean projection of the singular cases -- and that the module holds no arithmetic of the method
(it must not import the oracle or the binding's solver)."""
import ast
import os

import numpy as np

from paper_1909_05423_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shapes_and_spacings_follow_baseline_json():
    w1 = wl.config1("uniform")
    assert w1.shape == (32, 32, 32) and w1.bc == (wl.P, wl.P, wl.D) and np.allclose(w1.h, 1 / 32)
    w3 = wl.config3(8)
    assert w3.shape == (32, 64, 64) and w3.bc == (wl.P, wl.P, wl.N)
    assert np.allclose(w3.h, (1 / 64, 1 / 64, 1 / 32))
    w5 = wl.config5(scale=16)
    nz, ny, nx = w5.shape
    assert (nx, ny, nz) == (128, 128, 8) and w5.bc == (wl.N, wl.N, wl.D)
    assert np.isclose(w5.h[2], 4 * w5.h[0])                      # dz = 4 dx


def test_paper_pencils():
    w = wl.paper_pencil("PPN", nxy=16, nz=512)                   # small sibling of 64 x 64 x 16384
    assert w.shape == (512, 16, 16) and np.allclose(w.h, 1 / 16)   # cubic cells
    assert abs(w.f.mean()) < 1e-14                               # singular: projected to zero mean
    d = wl.paper_pencil("PPD", nxy=16, nz=512)
    assert abs(d.f.mean()) > 1e-6                                # not singular: left as drawn


def test_generators_are_seeded():
    a, b = wl.config2("NNN", "normal", n=16), wl.config2("NNN", "normal", n=16)
    assert np.array_equal(a.f, b.f)
    assert not np.array_equal(a.f, wl.config2("PPP", "normal", n=16).f)
    assert wl.seed_for(3, 0) == 190905423 + 300


def test_module_imports_nothing_of_the_method():
    src = open(os.path.join(ROOT, "paper_1909_05423_b200", "workloads.py")).read()
    mods = set()
    for node in ast.walk(ast.parse(src)):
        if isinstance(node, ast.Import):
            mods.update(a.name.split(".")[0] for a in node.names)
        elif isinstance(node, ast.ImportFrom) and node.module:
            mods.add(node.module.split(".")[0])
    assert mods <= {"__future__", "dataclasses", "numpy"}, mods
