"""GPU tests of the C-ABI contract: aliasing, plan reuse, determinism, streams, host solve,
error codes, profiling hooks."""
import ctypes

import numpy as np
import pytest

from oracle import poisson_oracle as po
from paper_1909_05423_b200 import workloads as wl
from gpu_util import TOL, gpu_solve, rel_err

pytestmark = pytest.mark.gpu


def test_in_place_equals_out_of_place_and_f_untouched():
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config2("PPN", "normal", n=64)
    plan = pp.Plan(64, 64, 64, *w.h, w.bc)
    f = torch.from_numpy(w.f).cuda()
    f0 = f.clone()
    u = plan.solve(f)
    torch.cuda.synchronize()
    assert torch.equal(f, f0)
    g = f.clone()
    plan.solve(g, g)
    torch.cuda.synchronize()
    assert torch.equal(g, u)                      # bitwise: same kernels, same order
    assert rel_err(u.cpu().numpy(), po.solve(w.f, w.h, w.bc)) <= TOL
    plan.destroy()


def test_plan_reuse_and_determinism():
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config2("NND", "normal", n=64)
    plan = pp.Plan(64, 64, 64, *w.h, w.bc)
    f = torch.from_numpy(w.f).cuda()
    outs = [plan.solve(f).clone() for _ in range(4)]
    torch.cuda.synchronize()
    for o in outs[1:]:
        assert torch.equal(o, outs[0])
    f2 = torch.from_numpy(wl.random_uniform(w.shape, 5)).cuda()
    u2 = plan.solve(f2)
    assert rel_err(u2.cpu().numpy(), po.solve(f2.cpu().numpy(), w.h, w.bc)) <= TOL
    plan.destroy()


def test_non_default_stream_is_ordered():
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config1("uniform")
    plan = pp.Plan(32, 32, 32, *w.h, w.bc)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        f = torch.from_numpy(w.f).cuda(non_blocking=False)
        f.mul_(2.0)                                # queued on s before the solve
        u = plan.solve(f)
        u.mul_(0.5)                                # queued on s after the solve
    s.synchronize()
    assert rel_err(u.cpu().numpy(), po.solve(w.f, w.h, w.bc)) <= TOL
    plan.destroy()


def test_host_solve():
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config2("PPD", "normal", n=32)
    plan = pp.Plan(32, 32, 32, *w.h, w.bc)
    before = plan.workspace_bytes
    fh = torch.from_numpy(w.f).pin_memory()
    uh = torch.empty_like(fh).pin_memory()
    plan.solve_host(fh, uh)
    assert plan.workspace_bytes == before + w.f.nbytes
    assert rel_err(uh.numpy(), po.solve(w.f, w.h, w.bc)) <= TOL
    plan.destroy()


def test_profiling_hooks():
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config1("uniform")
    plan = pp.Plan(32, 32, 32, *w.h, w.bc)
    f = torch.from_numpy(w.f).cuda()
    with pytest.raises(pp.PittPackError):
        plan.last_kernel_ms()                     # nothing recorded yet
    plan.set_profiling(True)
    plan.solve(f)
    ms = plan.last_kernel_ms()
    assert list(ms) == list(pp.KERNEL_NAMES) and all(v > 0 for v in ms.values())
    plan.destroy()


def test_error_codes_on_device():
    import torch
    import paper_1909_05423_b200 as pp
    st, h = pp.pp_plan_create(32, 32, 32, 0.1, 0.1, 0.1, 0, 0, 2)
    assert st == 0 and h
    f = torch.zeros(32 * 32 * 32 + 8, dtype=torch.float64, device="cuda")
    n = 32 * 32 * 32
    assert pp.pp_solve(h, 0, f.data_ptr()) == 5                               # NULL
    assert pp.pp_solve(0, f.data_ptr(), f.data_ptr()) == 5
    assert pp.pp_solve(h, f.data_ptr() + 8, f.data_ptr() + 8) == 1            # misaligned
    assert pp.pp_solve(h, f.data_ptr(), f.data_ptr() + 64) == 1               # partial overlap
    assert pp.pp_solve(h, f.data_ptr(), f.data_ptr()) == 0                    # exact alias is fine
    torch.cuda.synchronize()
    assert pp.pp_plan_destroy(h) == 0
    assert pp.pp_plan_destroy(0) == 0
    del n


@pytest.mark.parametrize("case", ["cfg1", "fused128", "long768", "long768-singular"])
def test_pp_solve_is_graph_capturable(case):
    """pp_solve never allocates and never synchronises (include/pittpack_b200.h), so a solve can be
    captured into a CUDA graph and replayed -- what a time-stepping caller does with small grids,
    where five launches cost more than the kernels (config 1: launch-latency bound)."""
    import torch
    import paper_1909_05423_b200 as pp
    if case == "cfg1":
        w = wl.config1("uniform")
    elif case == "fused128":
        w = wl.config2("PPN", "normal")
    else:
        shape = (768, 8, 16)
        combo = "NNN" if case.endswith("singular") else "NND"     # singular: the zero-mode kernel forks onto the side stream
        f0 = wl.random_normal(shape, 3, zero_mean=True)
        w = wl.Workload(case, shape, (1.0 / 16, 1.0 / 8, 1.0 / 8), wl.parse_bc(combo), f0)
    nz, ny, nx = w.shape
    plan = pp.Plan(nx, ny, nz, *w.h, w.bc)
    if case == "fused128":
        plan.set_xy_fusion(True)
    f = torch.from_numpy(w.f).cuda()
    u = torch.empty_like(f)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        plan.solve(f, u)                            # warm-up outside capture (function attributes, lazy module load)
    s.synchronize()
    ref = u.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        plan.solve(f, u)
    u.zero_()
    g.replay()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(u, ref)
    assert rel_err(u.cpu().numpy(), po.solve(w.f, w.h, w.bc)) <= TOL
    plan.destroy()


@pytest.mark.parametrize("combo,shape", [("PPN", (64, 16, 32)), ("NNN", (40, 8, 16)), ("PPP", (64, 16, 16)),
                                         ("NNP", (17, 8, 16)), ("PPN", (768, 8, 16))])
def test_pinned_plane_null_space(combo, shape):
    """The paper's own convention for singular problems: the mean of the z = 0 plane is kept
    at zero.  It differs from the zero-mean solution (the oracle's, R11) by a constant only."""
    import torch
    import paper_1909_05423_b200 as pp
    bc = wl.parse_bc(combo)
    nz, ny, nx = shape
    h = (1.0 / nx, 1.0 / ny, 2.0 / nz)
    f = wl.random_normal(shape, 900 + nz, zero_mean=True)
    ref = po.solve(f, h, bc)
    plan = pp.Plan(nx, ny, nz, *h, bc)
    plan.set_null_space("pin_plane0")
    u = plan.solve(torch.from_numpy(f).cuda()).cpu().numpy()
    assert abs(u[0].mean()) <= 1e-13 * np.abs(u).max()
    assert rel_err(u, ref - ref[0].mean()) <= TOL
    plan.set_null_space("zero_mean")
    u0 = plan.solve(torch.from_numpy(f).cuda()).cpu().numpy()
    assert rel_err(u0, ref) <= TOL
    plan.destroy()


def test_fold_dirichlet_faces_matches_the_oracle():
    """pp_fold_dirichlet against oracle.fold_dirichlet: bit-exact (one multiply, one subtract),
    all six faces at once on a non-cubic grid, then the solve of the folded source; and the refusal of a
    face on a non-Dirichlet axis."""
    import torch
    import paper_1909_05423_b200 as pp
    nz, ny, nx = 12, 16, 32
    h = (0.05, 0.04, 0.07)
    rng = np.random.default_rng(5)
    f = rng.standard_normal((nz, ny, nx))
    faces = {("x", 0): rng.standard_normal((nz, ny)), ("x", 1): rng.standard_normal((nz, ny)),
             ("y", 0): rng.standard_normal((nz, nx)), ("y", 1): rng.standard_normal((nz, nx)),
             ("z", 0): rng.standard_normal((ny, nx)), ("z", 1): rng.standard_normal((ny, nx))}
    bc = wl.parse_bc("DDD")
    ref_f = po.fold_dirichlet(f, h, bc, faces)
    plan = pp.Plan(nx, ny, nz, *h, bc)
    ft = torch.from_numpy(f).cuda()
    plan.fold_dirichlet(ft, {k: torch.from_numpy(v).cuda() for k, v in faces.items()})
    torch.cuda.synchronize()
    assert np.array_equal(ft.cpu().numpy(), ref_f)
    u = plan.solve(ft)
    assert rel_err(u.cpu().numpy(), po.solve(ref_f, h, bc)) <= TOL
    plan.destroy()
    plan = pp.Plan(nx, ny, nz, *h, wl.parse_bc("PDD"))
    with pytest.raises(pp.PittPackError):
        plan.fold_dirichlet(ft, {("x", 0): torch.zeros(nz, ny, dtype=torch.float64, device="cuda")})
    plan.fold_dirichlet(ft, {("z", 1): torch.zeros(ny, nx, dtype=torch.float64, device="cuda")})
    plan.destroy()


def test_host_batch_pipeline():
    """pp_solve_host_batch: five right-hand sides through a ring of three staging buffers; every solution
    equals the one-at-a-time host solve bit for bit."""
    import torch
    import paper_1909_05423_b200 as pp
    w = wl.config2("PPN", "normal", n=64)
    plan = pp.Plan(64, 64, 64, *w.h, w.bc)
    fb = torch.stack([torch.from_numpy(wl.random_normal(w.shape, 40 + i, zero_mean=True)) for i in range(5)]).pin_memory()
    ub = torch.empty_like(fb).pin_memory()
    plan.solve_host_batch(fb, ub)
    one = torch.empty(w.shape, dtype=torch.float64).pin_memory()
    for i in range(5):
        plan.solve_host(fb[i].contiguous().pin_memory(), one)
        assert torch.equal(ub[i], one), i
    assert rel_err(ub[4].numpy(), po.solve(fb[4].numpy(), w.h, w.bc)) <= TOL
    plan.solve_host_batch(fb[:2], ub[:2])              # shorter than the ring
    plan.destroy()


@pytest.mark.parametrize("shape,combo", [((32, 32, 32), "PPD"), ((12, 48, 96), "NNN"), ((7, 16, 64), "DPN"), ((3, 1024, 8), "PNP"),
                                         ((256, 8, 8), "NNN"), ((40, 8, 16), "PPP")])
def test_solve_batch_is_the_solves_one_by_one(shape, combo):
    """pp_solve_batch: the transforms of all right-hand sides in one launch per pass, the z solves one by one -- bit-identical
    to separate pp_solve calls (singular grids: every right-hand side gets its own zero-mode fix), out of place and in place."""
    import numpy as np
    import torch
    import paper_1909_05423_b200 as pp
    from paper_1909_05423_b200 import workloads as wl
    bc = wl.parse_bc(combo)
    nz, ny, nx = shape
    h = (1.0 / nx, 0.7 / ny, 1.3 / nz)
    nb = 3
    f = np.stack([wl.random_normal(shape, 900 + i, zero_mean=False) for i in range(nb)])
    plan = pp.Plan(nx, ny, nz, *h, bc)
    ft = torch.from_numpy(f).cuda()
    one = torch.stack([plan.solve(ft[i].contiguous()) for i in range(nb)])
    ub = plan.solve_batch(ft)
    torch.cuda.synchronize()
    assert torch.equal(one, ub)
    g = ft.clone()
    plan.solve_batch(g, g)
    torch.cuda.synchronize()
    assert torch.equal(one, g)
    with pytest.raises(ValueError):
        plan.solve_batch(ft[0])
    plan.destroy()


@pytest.mark.parametrize("nb", [65, 130])
def test_solve_batch_beyond_one_z_launch(nb):
    """More right-hand sides than one launch of the batched z kernel takes (64, Z_MAX_BATCH in csrc/pp_zshape.h): every
    solution against the oracle, and bit-identical to a pp_solve of its own."""
    import numpy as np
    import torch
    import paper_1909_05423_b200 as pp
    from oracle import poisson_oracle as po
    from paper_1909_05423_b200 import workloads as wl
    shape, bc = (32, 32, 32), wl.parse_bc("PPN")                    # singular: every grid gets its own zero-mode line
    h = (1.0 / 32, 0.7 / 32, 1.3 / 32)
    f = np.stack([wl.random_normal(shape, 2000 + i, zero_mean=False) for i in range(nb)])
    plan = pp.Plan(32, 32, 32, *h, bc)
    ft = torch.from_numpy(f).cuda()
    ub = plan.solve_batch(ft)
    torch.cuda.synchronize()
    got = ub.cpu().numpy()
    for i in range(nb):
        assert rel_err(got[i], po.solve(f[i], h, bc)) <= TOL, i
    for i in (0, 63, 64, nb - 1):
        assert torch.equal(plan.solve(ft[i].contiguous()), ub[i]), i
    plan.destroy()


@pytest.mark.parametrize("shape,combo", [((768, 8, 8), "PPP"), ((768, 128, 256), "NND"), ((768, 128, 256), "NNN"), ((512, 16, 8), "PPN")])
def test_solve_batch_on_long_lines(shape, combo):
    """Three right-hand sides where the z solve is not the one-CTA kernel: the two-level partition (8 x 8 x 768, cyclic;
    8 x 16 x 512 takes the one-CTA kernel with 64 rows per thread) and the cluster kernel (256 x 128 x 768), each against
    the oracle."""
    import numpy as np
    import torch
    import paper_1909_05423_b200 as pp
    from oracle import poisson_oracle as po
    from paper_1909_05423_b200 import workloads as wl
    bc = wl.parse_bc(combo)
    nz, ny, nx = shape
    h = (1.0 / nx, 0.7 / ny, 1.3 / nz)
    f = np.stack([wl.random_normal(shape, 3000 + i, zero_mean=False) for i in range(3)])
    plan = pp.Plan(nx, ny, nz, *h, bc)
    ft = torch.from_numpy(f).cuda()
    ub = plan.solve_batch(ft)
    torch.cuda.synchronize()
    got = ub.cpu().numpy()
    for i in range(3):
        assert rel_err(got[i], po.solve(f[i], h, bc)) <= TOL, i
        assert torch.equal(plan.solve(ft[i].contiguous()), ub[i]), i
    plan.destroy()


@pytest.mark.parametrize("shape,combo,nb", [((8, 8, 8), "NNN", 8200), ((256, 4, 4), "PPD", 257), ((16384, 4, 4), "DDN", 5)])
def test_solve_batch_taller_than_one_grid(shape, combo, nb):
    """nz * nbatch > 65535 planes: more than the y extent of one launch grid (the y passes put a plane on blockIdx.y), so
    the stack is solved in groups of floor(65535 / nz) grids.  Sampled solutions against the oracle -- the last grid of a
    group, the first of the next, the very last -- and the whole stack against the same stack solved in two halves."""
    import numpy as np
    import torch
    import paper_1909_05423_b200 as pp
    from oracle import poisson_oracle as po
    from paper_1909_05423_b200 import workloads as wl
    bc = wl.parse_bc(combo)
    nz, ny, nx = shape
    assert nz * nb > 65535
    h = (1.0 / nx, 0.7 / ny, 1.3 / nz) if nz <= 256 else (0.02, 0.03, 0.025)    # long lines: keep dz / dx of order one
    rng = np.random.default_rng(4000 + nb)
    f = rng.standard_normal((nb,) + shape)
    plan = pp.Plan(nx, ny, nz, *h, bc)
    ft = torch.from_numpy(f).cuda()
    ub = plan.solve_batch(ft)
    torch.cuda.synchronize()
    group = 65535 // nz
    for i in sorted({0, group - 1, group, min(2 * group, nb - 1), nb - 1}):
        assert rel_err(ub[i].cpu().numpy(), po.solve(f[i], h, bc)) <= TOL, i
    half = nb // 2
    two = torch.cat([plan.solve_batch(ft[:half].contiguous()), plan.solve_batch(ft[half:].contiguous())])
    torch.cuda.synchronize()
    assert torch.equal(two, ub)
    plan.destroy()
