"""GPU parity of the plane-wise fused x+y kernels (include/pittpack_b200.h, pp_plan_set_xy_fusion):
same tiles, same arithmetic, different schedule -- the result must be bit-identical to the
five-kernel path and match the oracle to 1e-11."""
import numpy as np
import pytest

from oracle import poisson_oracle as po
from paper_1909_05423_b200 import workloads as wl
from gpu_util import TOL, rel_err

pytestmark = pytest.mark.gpu


def solve(f, h, bc, fusion, in_place=False):
    import torch
    import paper_1909_05423_b200 as pp
    nz, ny, nx = f.shape
    plan = pp.Plan(nx, ny, nz, h[0], h[1], h[2], bc)
    plan.set_xy_fusion(fusion)
    ft = torch.from_numpy(np.ascontiguousarray(f)).cuda()
    ut = plan.solve(ft, ft if in_place else None)
    torch.cuda.synchronize()
    u = ut.cpu().numpy()
    plan.destroy()
    return u


@pytest.mark.parametrize("n", [128, 256, 512])
@pytest.mark.parametrize("combo", ["PPN", "NND", "DDD", "PNP", "DPN", "NNN"])
def test_fused_is_bit_identical_and_matches_oracle(n, combo):
    bc = wl.parse_bc(combo)
    nz = {128: 37, 256: 12, 512: 7}[n]          # several lags' worth of planes at the small sizes
    shape = (nz, n, n)
    h = (1.0 / n, 0.9 / n, 1.0 / 16)
    f = wl.random_normal(shape, 500 + n, zero_mean=all(b in (0, 1) for b in bc))
    u0 = solve(f, h, bc, False)
    u1 = solve(f, h, bc, True)
    assert np.array_equal(u0, u1), (n, combo, float(np.max(np.abs(u0 - u1))))
    if n <= 256:
        ref = po.solve(f, h, bc)
        assert rel_err(u1, ref) <= TOL


def test_fused_in_place_and_repeated():
    """In place (u == f), and the same plan solving twice (the scheduler's counters are reset per launch)."""
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config2("PPN", "normal")
    nz, ny, nx = w.shape
    ref = po.solve(w.f, w.h, w.bc)
    assert rel_err(solve(w.f, w.h, w.bc, True, in_place=True), ref) <= TOL
    plan = pp.Plan(nx, ny, nz, *w.h, w.bc)
    plan.set_xy_fusion(True)
    f = torch.from_numpy(w.f).cuda()
    for _ in range(3):
        u = plan.solve(f)
    torch.cuda.synchronize()
    assert rel_err(u.cpu().numpy(), ref) <= TOL
    plan.destroy()


def test_fusion_refused_where_it_does_not_apply():
    import paper_1909_05423_b200 as pp
    for nx, ny in ((64, 64), (256, 128), (2048, 2048), (384, 384)):
        plan = pp.Plan(nx, ny, 4, 0.1, 0.1, 0.1, "PPN")
        with pytest.raises(pp.PittPackError):
            plan.set_xy_fusion(True)
        plan.set_xy_fusion(False)
        plan.destroy()


# ---- x/y slab pipeline on two streams (pp_plan_set_xy_pipeline): plain launches, same kernels, same arithmetic
@pytest.mark.parametrize("shape,combo,planes", [((37, 128, 128), "PPN", 8), ((37, 128, 128), "NND", 5), ((12, 96, 48), "DPN", 1),
                                                ((40, 64, 256), "NNN", 16), ((9, 1024, 16), "DDD", 4), ((6, 32, 32), "PPP", 6)])
def test_pipelined_is_bit_identical(shape, combo, planes):
    """Ragged last slab, one plane per slab, a slab as large as the grid (= off), long y lines; in place and out of place;
    the plan solves three times in a row (the slab events are re-recorded)."""
    import torch
    import paper_1909_05423_b200 as pp
    bc = wl.parse_bc(combo)
    nz, ny, nx = shape
    h = (1.0 / nx, 0.9 / ny, 1.0 / 16)
    f = wl.random_normal(shape, 700 + nz, zero_mean=all(b in (0, 1) for b in bc))
    u0 = solve(f, h, bc, False)
    plan = pp.Plan(nx, ny, nz, *h, bc)
    plan.set_xy_pipeline(planes)
    ft = torch.from_numpy(f).cuda()
    for _ in range(3):
        u1 = plan.solve(ft)
    torch.cuda.synchronize()
    assert np.array_equal(u0, u1.cpu().numpy())
    g = ft.clone()
    plan.solve(g, g)
    torch.cuda.synchronize()
    assert np.array_equal(u0, g.cpu().numpy())
    plan.set_xy_pipeline(0)
    assert np.array_equal(u0, plan.solve(ft).cpu().numpy())
    plan.destroy()


def test_pipelined_under_graph_capture():
    """pp_solve with the pipeline on forks onto the plan's second stream and joins again: capturable."""
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config2("PPN", "normal", n=64)
    nz, ny, nx = w.shape
    plan = pp.Plan(nx, ny, nz, *w.h, w.bc)
    plan.set_xy_pipeline(16)
    f = torch.from_numpy(w.f).cuda()
    u = torch.empty_like(f)
    plan.solve(f, u)                                      # first solve outside the capture (kernel attributes)
    torch.cuda.synchronize()
    u.zero_()
    g = torch.cuda.CUDAGraph()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        with torch.cuda.graph(g, stream=st):
            plan.solve(f, u, stream=st)
    g.replay()
    torch.cuda.synchronize()
    ref = po.solve(w.f, w.h, w.bc)
    assert rel_err(u.cpu().numpy(), ref) <= TOL
    plan.destroy()
