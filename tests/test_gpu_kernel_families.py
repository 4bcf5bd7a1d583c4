"""Small solves that exercise every kernel family once, each compared with the oracle (1e-11): BASELINE.json config 1
(32^3 PPD); a 128 x 128 x 32 PPN grid with the x+y fusion kernel (ticket / acquire scheduler) and with the two-stream
x/y slab pipeline; a 64 x 32 x 768 NNN grid (two-level z solve with the singular line forked onto the side stream);
48 x 96 x 40 (mixed-radix lengths, two-sweep z); periodic z on one and two levels; long x and y lines; a slab
decomposition over two virtual ranks.

Collected by `pytest -m gpu`.  Run as a plain program (`python tests/test_gpu_kernel_families.py`) it goes through the same
cases in one process: the form a memory checker wants (profiles/r02_sanitizer.md; the file was tests/sanitizer_cases.py then).
"""
from __future__ import annotations

import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_1909_05423_b200 as pp                      # noqa: E402
from paper_1909_05423_b200 import workloads as wl       # noqa: E402
from oracle import poisson_oracle as po                 # noqa: E402


def check(name, u, f, h, bc):
    ref = po.solve(f, h, bc)
    err = float(np.max(np.abs(u.cpu().numpy() - ref)) / np.max(np.abs(ref)))
    print(f"{name}: max rel err {err:.2e}", flush=True)
    assert err <= 1e-11, (name, err)


def solve_case(name, shape, bc, h=None, fusion=False, pipeline=0, seed=5):
    nz, ny, nx = shape
    h = h or (1.0 / nx, 1.0 / ny, 1.0 / nz)
    bct = wl.parse_bc(bc)
    f = wl.random_normal(shape, seed, zero_mean=all(b != 2 for b in bct))
    plan = pp.Plan(nx, ny, nz, *h, bc)
    if fusion:
        plan.set_xy_fusion(True)
    if pipeline:
        plan.set_xy_pipeline(pipeline)
    import torch
    u = plan.solve(torch.from_numpy(f).cuda())
    torch.cuda.synchronize()
    check(name, u, f, h, bct)
    plan.destroy()


CASES = [
    ("128x128x32 PPN fused", (32, 128, 128), "PPN", dict(fusion=True)),
    ("128x128x32 PPN pipelined", (32, 128, 128), "PPN", dict(pipeline=8)),
    ("64x32x768 NNN two-level z", (768, 32, 64), "NNN", dict(h=(1 / 64, 1 / 64, 1 / 64))),
    ("48x96x40 NDP mixed radix", (40, 96, 48), "NDP", {}),
    ("32x32x64 PPP cyclic partition", (64, 32, 32), "PPP", {}),
    ("32x32x512 DNP two-level cyclic", (512, 32, 32), "DNP", dict(h=(1 / 32, 1 / 32, 1 / 32))),
    ("1024x8x8 DDD long x", (8, 8, 1024), "DDD", {}),
    ("8x2048x8 NND long y", (8, 2048, 8), "NND", {}),
]


@pytest.mark.gpu
@pytest.mark.parametrize("name,shape,bc,kw", CASES, ids=[c[0].replace(" ", "_") for c in CASES])
def test_kernel_family(name, shape, bc, kw):
    solve_case(name, shape, bc, **kw)


@pytest.mark.gpu
def test_config1_and_two_virtual_ranks():
    config1_and_slab()


def config1_and_slab():
    import torch
    w = wl.config1("uniform")
    nz, ny, nx = w.shape
    plan = pp.Plan(nx, ny, nz, *w.h, w.bc)
    u = plan.solve(torch.from_numpy(w.f).cuda())
    torch.cuda.synchronize()
    check("config 1", u, w.f, w.h, w.bc)
    plan.destroy()
    from paper_1909_05423_b200 import slab
    shape, bc = (16, 32, 32), "PNN"
    f = wl.random_normal(shape, 9, zero_mean=True)
    sp = slab.VirtualRanks(2, 32, 32, 16, 1 / 32, 1 / 32, 1 / 16, bc)
    u = sp.solve(torch.from_numpy(f).cuda())
    torch.cuda.synchronize()
    check("slab decomposition, 2 virtual ranks", u, f, (1 / 32, 1 / 32, 1 / 16), wl.parse_bc(bc))
    sp.destroy()


if __name__ == "__main__":
    config1_and_slab()
    for case in CASES:
        solve_case(case[0], case[1], case[2], **case[3])
    print("all cases passed")
