"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the
same seeded inputs.  Bar: max|u_gpu - u_ref| / max|u_ref| <= 1e-11 (north_star)."""
import itertools

import numpy as np
import pytest

from oracle import poisson_oracle as po
from paper_1909_05423_b200 import workloads as wl
from gpu_util import TOL, gpu_solve, rel_err

pytestmark = pytest.mark.gpu

ALL27 = ["".join(c) for c in itertools.product("PND", repeat=3)]


def check(w: wl.Workload, tol=TOL, **kw):
    u = gpu_solve(w.f, w.h, w.bc, **kw)
    ref = po.solve(w.f, w.h, w.bc)
    e = rel_err(u, ref)
    assert e <= tol, (w.name, e)
    return u, ref


@pytest.mark.parametrize("combo", ALL27)
@pytest.mark.parametrize("shape", [(12, 8, 16), (5, 32, 8), (40, 16, 64)], ids=lambda s: "x".join(map(str, s[::-1])))
def test_all_27_combos_small(combo, shape):
    """Every boundary-condition combination; non-cubic, nz not a power of two, anisotropic spacing."""
    bc = wl.parse_bc(combo)
    nz, ny, nx = shape
    h = (1.0 / nx, 0.7 / ny, 1.3 / nz)
    f = wl.random_uniform(shape, 7 + ALL27.index(combo))
    check(wl.Workload(f"{combo}-{shape}", shape, h, bc, f))


@pytest.mark.parametrize("n", [4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048])
@pytest.mark.parametrize("axis", ["x", "y"])
@pytest.mark.parametrize("bc_t", "PND")
def test_every_fft_length(n, axis, bc_t):
    """Each supported transform length on each axis, each transform type, ragged tiles."""
    other = 4 if n >= 512 else 8
    nx, ny = (n, other) if axis == "x" else (other, n)
    nz = 3
    combo = (bc_t + "N" + "D") if axis == "x" else ("D" + bc_t + "N")
    shape = (nz, ny, nx)
    h = (1.0 / nx, 1.0 / ny, 0.5)
    f = wl.random_uniform(shape, n + (0 if axis == "x" else 1))
    check(wl.Workload(f"len{n}{axis}{bc_t}", shape, h, wl.parse_bc(combo), f))


@pytest.mark.parametrize("n", [48, 96, 192, 384, 768, 1536, 80, 160, 320, 640, 1280])
@pytest.mark.parametrize("axis", ["x", "y"])
@pytest.mark.parametrize("bc_t", "PND")
def test_every_mixed_radix_length(n, axis, bc_t):
    """3*2^k and 5*2^k lengths (the 48-multiples of the paper's weak-scaling grids):
    prime-factor first stage + radix-4 stages, each transform type on each axis."""
    other = 4 if n >= 512 else 8
    nx, ny = (n, other) if axis == "x" else (other, n)
    nz = 3
    combo = (bc_t + "N" + "D") if axis == "x" else ("D" + bc_t + "N")
    shape = (nz, ny, nx)
    h = (1.0 / nx, 1.0 / ny, 0.5)
    f = wl.random_uniform(shape, 3 * n + (0 if axis == "x" else 1))
    check(wl.Workload(f"len{n}{axis}{bc_t}", shape, h, wl.parse_bc(combo), f))


@pytest.mark.parametrize("combo", ALL27)
def test_all_27_combos_on_a_48_multiple(combo):
    """48 x 96 x 40: the paper's 48-multiple grid shape, every boundary-condition combination."""
    bc = wl.parse_bc(combo)
    shape = (40, 96, 48)
    h = (1.0 / 48, 1.0 / 96, 1.0 / 40)
    f = wl.random_normal(shape, 48 + ALL27.index(combo), zero_mean=all(b in (0, 1) for b in bc))
    check(wl.Workload(f"mixed-{combo}", shape, h, bc, f))


def test_config1_both_variants():
    for variant in ("mms", "uniform"):
        w = wl.config1(variant)
        u, ref = check(w)
        if variant == "mms":       # eigenfunction: second-order accurate against the analytic solution
            assert np.max(np.abs(u - w.u_exact)) < 5e-3


@pytest.mark.parametrize("combo", wl.CONFIG2_COMBOS)
@pytest.mark.parametrize("variant", ["mms", "normal"])
def test_config2_128cubed(combo, variant):
    check(wl.config2(combo, variant))


@pytest.mark.parametrize("combo", ["PPN", "NNP", "DPD", "PDP", "NPN"])
def test_tile_boundaries_and_long_z(combo):
    """Several x tiles, several y tiles, nz spanning several checkpoint blocks with a ragged tail."""
    shape = (67, 64, 128)
    h = (1.0 / 128, 1.0 / 64, 1.0 / 67)
    bc = wl.parse_bc(combo)
    f = wl.random_normal(shape, 31, zero_mean=all(b in (0, 1) for b in bc))
    check(wl.Workload(f"tiles-{combo}", shape, h, bc, f))


def test_nz_extremes():
    for nz in (2, 3, 16, 17, 1025):
        for combo in ("PPN", "NDD", "DNP"):
            shape = (nz, 8, 16)
            f = wl.random_uniform(shape, nz)
            check(wl.Workload(f"nz{nz}-{combo}", shape, (0.1, 0.1, 0.1), wl.parse_bc(combo), f))


def test_config3_scaled_siblings():
    for scale in (8, 4, 2):
        check(wl.config3(scale))


def test_config4_and_5_scaled():
    check(wl.config4(64))
    check(wl.config4(128, twin=True))
    check(wl.config5(scale=8))


@pytest.mark.parametrize("combo", ALL27)
def test_second_order_convergence_on_gpu(combo):
    """MMS error ratio 4 +- 0.3 on grid halving for every BC combination (north_star)."""
    bc = wl.parse_bc(combo)
    errs = []
    for n in (16, 32, 64):
        shape, h = (n, n, n), (1.0 / n,) * 3
        f, u, _ = wl.mms(shape, h, bc)
        uh = gpu_solve(f, h, bc)
        if all(b in (0, 1) for b in bc):
            u = u - u.mean()
        errs.append(float(np.sqrt(np.mean((uh - u) ** 2))))
    for coarse, fine in zip(errs[:-1], errs[1:]):
        assert abs(coarse / fine - 4.0) <= 0.3, errs


@pytest.mark.parametrize("ny", [1024, 1280, 1536, 2048])
@pytest.mark.parametrize("nx,combo", [(8, "PPN"), (48, "PPP"), (8, "PNN"), (16, "NPD"), (48, "PDD"), (4, "NNN")])
def test_tma_staged_y_tiles(ny, nx, combo):
    """The y passes of 1024 rows and more fetch their tiles through tensor maps (ypass_*_tma_kernel):
    complex columns (x and y periodic), real pairs, every y transform type, tiles that hang over the last column
    (nxh = 2 with four-column tiles), three planes (the forward pass walks them in reverse); out of place and in place."""
    bc = wl.parse_bc(combo)
    shape = (3, ny, nx)
    h = (1.0 / nx, 1.0 / ny, 0.25)
    f = wl.random_normal(shape, ny + nx, zero_mean=all(b in (0, 1) for b in bc))
    w = wl.Workload(f"tma{ny}x{nx}{combo}", shape, h, bc, f)
    u, ref = check(w)
    u2 = gpu_solve(w.f, w.h, w.bc, in_place=True)
    assert np.array_equal(u, u2)


def test_tma_staged_under_graph_capture():
    """The tensor maps are built on the host at launch and passed by value: a captured solve replays correctly."""
    import torch
    import paper_1909_05423_b200 as pp
    shape, h, bc = (4, 1024, 16), (1.0 / 16, 1.0 / 1024, 0.25), wl.parse_bc("NDN")
    f = wl.random_normal(shape, 5, zero_mean=False)
    plan = pp.Plan(16, 1024, 4, *h, bc)
    ft = torch.from_numpy(f).cuda()
    u = torch.empty_like(ft)
    plan.solve(ft, u)
    torch.cuda.synchronize()
    u.zero_()
    g, st = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.stream(st):
        with torch.cuda.graph(g, stream=st):
            plan.solve(ft, u, stream=st)
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    assert rel_err(u.cpu().numpy(), po.solve(f, h, bc)) <= TOL
    plan.destroy()
