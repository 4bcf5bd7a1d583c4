"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

Every configuration is compared with the oracle element by element: config 3 (512x512x256, the headline)
by ``po.solve`` on the whole array; configs 4 and 5 (2^30 and 2^29 points) by the oracle's own functions
applied block by block on the host (tests/oracle_blocked.py -- the whole-array temporaries of ``po.solve`` would
need > 60 GB), a few minutes of host time each.  Kept beside them: the 7-point residual of eq. 3
 at 300 000 sampled cells (checker pinned on the CPU: tests/test_oracle_stencil.py) and, for the
eigenfunction twin of config 4, the closed-form discrete solution."""
import math

import numpy as np
import pytest

from oracle import poisson_oracle as po
from paper_1909_05423_b200 import workloads as wl
from gpu_util import TOL, rel_err
from oracle_blocked import oracle_solve_blocked, rel_err_blocked
from stencil_sampling import gather_torch, neighbour_table, sample_indices

pytestmark = pytest.mark.gpu

EPS = np.finfo(np.float64).eps


def test_config3_full_size_element_by_element():
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config3()
    nz, ny, nx = w.shape
    plan = pp.Plan(nx, ny, nz, *w.h, w.bc)
    f = torch.from_numpy(w.f).cuda()
    u = plan.solve(f)
    torch.cuda.synchronize()
    ug = u.cpu().numpy()
    plan.destroy()
    del f, u
    ref = po.solve(w.f, w.h, w.bc)
    e = rel_err(ug, ref)
    assert e <= TOL, e
    assert abs(ug.mean()) <= 1e-13 * np.max(np.abs(ug))          # zero-mean invariant


def residual_check(u, f, h, bc, seed):
    idx = sample_indices(tuple(u.shape), 300_000, seed)
    nb = gather_torch(u, neighbour_table(idx, tuple(u.shape), bc))   # ghost rules: NumPy, pinned on the CPU
    Au = po.stencil_at(nb, h)                                    # the oracle, one sampled cell at a time
    fs = f[idx]
    fmax = float(np.max(np.abs(fs)))
    normA = 4.0 * sum(1.0 / (v * v) for v in h)
    bound = max(1e-10 * fmax, 8 * EPS * normA * float(np.max(np.abs(nb[:, 0]))))     # DESIGN.md R24
    res = float(np.max(np.abs(Au - fs)))
    assert res <= bound, (res, bound)


def test_config5_full_size_sampled():
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config5()
    nz, ny, nx = w.shape
    plan = pp.Plan(nx, ny, nz, *w.h, w.bc)
    f = torch.from_numpy(w.f).cuda()
    u = plan.solve(f)
    torch.cuda.synchronize()
    residual_check(u, w.f, w.h, w.bc, seed=5)
    plan.destroy()


def config4_on_device(n, twin):
    """The config-4 recipe (workloads.config4) assembled on the device from its 1-D factor, so that
    the 8 GiB field never has to live in host memory."""
    import torch
    hh = 1.0 / n if twin else 1.0 / (n + 1)
    g = torch.from_numpy(np.sin(np.pi * wl.centres(n, hh))).cuda()
    f = (g[:, None, None] * g[None, :, None]) * g[None, None, :]
    f *= -3.0 * math.pi ** 2
    if not twin:
        gf = math.sin(math.pi * n * hh)
        c = 2.0 / (hh * hh)
        face = c * gf * (g[:, None] * g[None, :])
        f[:, :, n - 1] -= face
        f[:, n - 1, :] -= face
        f[n - 1, :, :] -= face
    return f, g, hh


def test_config4_device_recipe_matches_workloads():
    for twin in (False, True):
        f, _, _ = config4_on_device(32, twin)
        np.testing.assert_allclose(f.cpu().numpy(), wl.config4(32, twin).f, rtol=0, atol=1e-9)


@pytest.mark.parametrize("twin", [False, True])
def test_config4_full_size_sampled(twin):
    import torch
    import paper_1909_05423_b200 as pp
    n = 1024
    f, g, hh = config4_on_device(n, twin)
    bc = (2, 2, 2)
    h = (hh, hh, hh)
    plan = pp.Plan(n, n, n, hh, hh, hh, bc)
    u = plan.solve(f)
    torch.cuda.synchronize()
    idx = sample_indices((n, n, n), 300_000, seed=4)
    nb = gather_torch(u, neighbour_table(idx, (n, n, n), bc))
    k, j, i = (torch.from_numpy(v).cuda() for v in idx)
    fs = f[k, j, i].cpu().numpy()
    Au = po.stencil_at(nb, h)
    normA = 12.0 / (hh * hh)
    bound = max(1e-10 * float(np.max(np.abs(fs))), 8 * EPS * normA * float(np.max(np.abs(nb[:, 0]))))
    assert float(np.max(np.abs(Au - fs))) <= bound
    gs = g.cpu().numpy()
    u_exact = gs[idx[0]] * gs[idx[1]] * gs[idx[2]]
    if twin:
        # sin(pi x) is a discrete eigenfunction: u_h = u * 3 pi^2 / (3 (2/h)^2 sin^2(pi h / 2))   (Table 2)
        lam = 3.0 * (2.0 / hh) ** 2 * math.sin(math.pi * hh / 2.0) ** 2
        closed = u_exact * (3.0 * math.pi ** 2) / lam
        assert float(np.max(np.abs(nb[:, 0] - closed))) <= 1e-11
    else:
        assert float(np.max(np.abs(nb[:, 0] - u_exact))) <= 5e-6     # second-order accurate, h = 1/1025
    plan.destroy()


def host_memory_gib():
    with open("/proc/meminfo") as fh:
        for line in fh:
            if line.startswith("MemAvailable"):
                return int(line.split()[1]) / 2 ** 20
    return 0.0


def solve_to_host(f_dev, h, bc):
    """GPU solve through the C ABI (default plan: the launch configuration bench.py times), result on the host."""
    import torch
    import paper_1909_05423_b200 as pp
    nz, ny, nx = f_dev.shape
    plan = pp.Plan(nx, ny, nz, *h, bc)
    u = plan.solve(f_dev)
    torch.cuda.synchronize()
    ug = u.cpu().numpy()
    plan.destroy()
    return ug


def test_config5_full_size_element_by_element():
    """2048 x 2048 x 128 NND, every element against the oracle (block-wise driver: tests/oracle_blocked.py)."""
    import torch
    if host_memory_gib() < 14:
        pytest.skip("needs 14 GiB of host memory for the oracle's arrays")
    w = wl.config5()
    f = torch.from_numpy(w.f).cuda()
    ug = solve_to_host(f, w.h, w.bc)
    del f
    torch.cuda.empty_cache()
    ref = oracle_solve_blocked(w.f, w.h, w.bc)                    # in place: w.f now holds the oracle's u
    e = rel_err_blocked(ug, ref)
    assert e <= TOL, e


@pytest.mark.parametrize("twin", [False, True])
def test_config4_full_size_element_by_element(twin):
    """1024^3 DDD as written in BASELINE.json (h = 1/1025, folded faces) and its h = 1/1024 twin, every
    element against the oracle; the twin also against the closed-form discrete solution (Table 2)."""
    import torch
    if host_memory_gib() < 26:
        pytest.skip("needs 26 GiB of host memory for the oracle's arrays")
    n = 1024
    f, g, hh = config4_on_device(n, twin)
    bc, h = (2, 2, 2), (hh, hh, hh)
    fh = f.cpu().numpy()
    ug = solve_to_host(f, h, bc)
    del f
    torch.cuda.empty_cache()
    ref = oracle_solve_blocked(fh, h, bc)
    e = rel_err_blocked(ug, ref)
    assert e <= TOL, e
    if twin:
        gs = g.cpu().numpy()
        lam = 3.0 * (2.0 / hh) ** 2 * math.sin(math.pi * hh / 2.0) ** 2
        worst = 0.0
        for k0 in range(0, n, 16):
            closed = (gs[k0:k0 + 16, None, None] * gs[None, :, None] * gs[None, None, :]) * ((3.0 * math.pi ** 2) / lam)
            worst = max(worst, float(np.max(np.abs(ug[k0:k0 + 16] - closed))))
        assert worst <= 1e-11, worst
