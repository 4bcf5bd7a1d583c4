"""GPU parity of the two z-solve kernels (include/pittpack_b200.h, pp_plan_set_z_algorithm): the
partitioned register-resident solve and the two-sweep Thomas must each match the oracle to 1e-11
on the same seeded inputs, for every segment count the partitioned kernel supports."""
import numpy as np
import pytest

from oracle import poisson_oracle as po
from paper_1909_05423_b200 import workloads as wl
from gpu_util import TOL, gpu_solve, rel_err

pytestmark = pytest.mark.gpu

# nz -> (rows per thread, segments): 32 m (m <= 8), 64 m (m <= 8), 1024, 2048
PART_NZ = [32, 64, 96, 128, 160, 192, 224, 256, 320, 384, 448, 512, 1024, 2048]


@pytest.mark.parametrize("nz", PART_NZ)
@pytest.mark.parametrize("combo", ["PPN", "NND", "DDN", "NNN", "PDD", "PPP", "NDP", "DDP"])
def test_partition_matches_oracle(nz, combo):
    """Plane of 8 x 20-ish systems: ragged last CTA (the plane is not a multiple of 32 systems)."""
    bc = wl.parse_bc(combo)
    nx, ny = (8, 4) if nz >= 1024 else (8, 16)
    shape = (nz, ny, nx)
    h = (1.0 / nx, 0.8 / ny, 2.0 / nz)
    f = wl.random_normal(shape, 1000 + nz, zero_mean=all(b in (0, 1) for b in bc))
    ref = po.solve(f, h, bc)
    for alg in ("partition", "sweep"):
        u = gpu_solve(f, h, bc, z_algorithm=alg)
        e = rel_err(u, ref)
        assert e <= TOL, (alg, nz, combo, e)


@pytest.mark.parametrize("combo", ["PPN", "NNN", "DDD", "NDN", "PPP", "NNP"])
def test_partition_small_shift_modes(combo):
    """Strongly anisotropic spacing (dz << dx): |s| = dz^2 (lam_x/dx^2 + lam_y/dy^2) is tiny for the
    low modes, the pivots stay near -1 and the interface system is at its worst conditioned."""
    bc = wl.parse_bc(combo)
    shape = (256, 16, 32)
    h = (1.0 / 32, 1.0 / 16, 1.0 / 1024)
    f = wl.random_normal(shape, 77, zero_mean=all(b in (0, 1) for b in bc))
    ref = po.solve(f, h, bc)
    for alg in ("partition", "sweep"):
        e = rel_err(gpu_solve(f, h, bc, z_algorithm=alg), ref)
        assert e <= TOL, (alg, combo, e)


def test_partition_large_shift_modes():
    """dz >> dx: |b| is large, the leading minors grow like |b|^R (no overflow, no loss of accuracy)."""
    shape = (128, 32, 32)
    h = (1.0 / 2048, 1.0 / 2048, 1.0 / 16)
    for combo in ("PPN", "DDD", "PPP"):
        bc = wl.parse_bc(combo)
        f = wl.random_normal(shape, 78, zero_mean=all(b in (0, 1) for b in bc))
        ref = po.solve(f, h, bc)
        e = rel_err(gpu_solve(f, h, bc, z_algorithm="partition"), ref)
        assert e <= TOL, (combo, e)


def test_extreme_anisotropy_falls_back_to_the_sweep():
    """dz/dx = 256 with 64-row segments: the leading minors would reach |b|^64 ~ 1e360 and leave the fp64
    range, so the plan must not use the partitioned kernel there (and must still be right)."""
    import paper_1909_05423_b200 as pp
    shape = (1024, 8, 16)
    h = (1.0 / 4096, 1.0 / 4096, 1.0 / 16)
    bc = wl.parse_bc("NND")
    f = wl.random_uniform(shape, 11)
    ref = po.solve(f, h, bc)
    assert rel_err(gpu_solve(f, h, bc), ref) <= TOL
    plan = pp.Plan(16, 8, 1024, *h, bc)
    with pytest.raises(pp.PittPackError):
        plan.set_z_algorithm("partition")
    plan.destroy()
    # the same grid with 32-row segments (nz = 256) is inside the range
    shape = (256, 8, 16)
    f = wl.random_uniform(shape, 12)
    assert rel_err(gpu_solve(f, h, bc, z_algorithm="partition"), po.solve(f, h, bc)) <= TOL


def test_partition_refused_where_it_does_not_apply():
    import paper_1909_05423_b200 as pp
    for nz, combo in ((48, "PPN"), (800, "PPP"), (100, "DDD")):
        plan = pp.Plan(8, 8, nz, 0.1, 0.1, 0.1, combo)
        with pytest.raises(pp.PittPackError):
            plan.set_z_algorithm("partition")
        plan.set_z_algorithm("sweep")
        plan.set_z_algorithm("auto")
        plan.destroy()


# ---------------------------------------------------------------- long lines: two-level partition
@pytest.mark.parametrize("nz", [512 + 256, 1280, 2304, 4096])
@pytest.mark.parametrize("combo", ["PPN", "NND", "DDD", "NNN", "PPP", "NNP", "DNP"])
def test_two_level_partition_matches_oracle(nz, combo):
    """nz = 256 m that no single CTA holds: super-segments of 256 rows coupled by the interface
    kernel (periodic z: the chain of super-segments closes on itself).  The two-sweep kernel solves the
    same systems: both must match the oracle."""
    bc = wl.parse_bc(combo)
    shape = (nz, 4, 24 if False else 16)
    h = (1.0 / 16, 1.0 / 4, 1.0 / 8)
    f = wl.random_normal(shape, 2000 + nz, zero_mean=all(b in (0, 1) for b in bc))
    ref = po.solve(f, h, bc)
    for alg in ("partition", "sweep"):
        e = rel_err(gpu_solve(f, h, bc, z_algorithm=alg), ref)
        assert e <= TOL, (alg, nz, combo, e)


@pytest.mark.parametrize("combo", ["PPD", "PPN", "PPP", "NNP"])
def test_paper_pencil_shape(combo):
    """64 x 64 x 16384, the paper's per-GPU weak-scaling load: beyond the two-sweep
    kernel's range, solved by the two-level partition only."""
    w = wl.paper_pencil(combo)
    # Lines this long are ill-conditioned (cond(T) ~ nz^2 for the lowest modes): an fp64 Thomas sweep
    # is itself only good to ~1e-11 here, so the ground truth is the oracle with its z solve in
    # long double (oracle/poisson_oracle.py, zdtype; SURVEY.md 8(c) "precision hazards").
    ref = po.solve(w.f, w.h, w.bc, zdtype=np.longdouble)
    u = gpu_solve(w.f, w.h, w.bc)
    e = rel_err(u, ref)
    assert e <= TOL, (combo, e)
    e64 = rel_err(po.solve(w.f, w.h, w.bc), ref)
    print(f"pencil {combo}: gpu vs long-double oracle {e:.2e}; fp64 oracle vs long-double oracle {e64:.2e}")


def test_paper_pencil_48():
    """48 x 48 x 8192: mixed-radix transforms and the two-level z solve together."""
    w = wl.paper_pencil("PPN", nxy=48, nz=8192)
    ref = po.solve(w.f, w.h, w.bc, zdtype=np.longdouble)
    e = rel_err(gpu_solve(w.f, w.h, w.bc), ref)
    assert e <= TOL, e


@pytest.mark.parametrize("nz", [5000, 8200, 4097, 16383])
@pytest.mark.parametrize("combo", ["PPN", "NND", "PPP"])
def test_long_lines_of_any_length(nz, combo):
    """nz beyond 4096 that is not a multiple of 256 (the two-level partition does not take it): the two-sweep
    kernels with their checkpoint tables in shared memory.  Ground truth: the oracle with a long-double z solve."""
    bc = wl.parse_bc(combo)
    shape, h = (nz, 8, 16), (1.0 / 16, 1.0 / 8, 1.0 / 16)
    f = wl.random_normal(shape, 3000 + nz, zero_mean=all(b in (0, 1) for b in bc))
    ref = po.solve(f, h, bc, zdtype=np.longdouble)
    e = rel_err(gpu_solve(f, h, bc), ref)
    assert e <= TOL, (nz, combo, e)


def test_long_line_limits():
    import paper_1909_05423_b200 as pp
    for nz, combo, ok in ((8192, "PPN", True), (8192, "PPP", True), (8192 + 128, "PPN", True), (16384, "NNP", True),
                          (16385, "PPN", False), (32768, "PPD", False)):
        st, h = pp.binding.pp_plan_create(8, 8, nz, 0.1, 0.1, 0.1, *wl.parse_bc(combo))
        assert (st == 0) == ok, (nz, combo, st)
        if h:
            assert pp.binding.pp_plan_set_z_algorithm(h, pp.binding.PP_Z_SWEEP) == 0      # any nz has a two-sweep path
            want = 0 if nz % 256 == 0 else 2                                              # two-level: multiples of 256
            assert pp.binding.pp_plan_set_z_algorithm(h, pp.binding.PP_Z_PARTITION) == want
            pp.binding.pp_plan_destroy(h)


# ---- cluster kernel (PP_Z_CLUSTER): both levels of the long-line partition in one pass, super-segment interfaces
# exchanged through distributed shared memory (include/pittpack_b200.h)
@pytest.mark.parametrize("nz", [512, 768, 1024, 1280, 1536, 1792, 2048])
@pytest.mark.parametrize("combo", ["PPN", "NND", "DDN", "NNN", "PDD"])
def test_cluster_matches_oracle(nz, combo):
    """Forced on small planes: 4 x 4 lines (half of each CTA idle) or 16 x 4 (two clusters per line set)."""
    bc = wl.parse_bc(combo)
    shape = (nz, 4, 4) if (nz // 256) % 2 else (nz, 4, 16)
    h = (1.0 / shape[2], 0.8 / 4, 2.0 / nz)
    f = wl.random_normal(shape, 2000 + nz, zero_mean=all(b in (0, 1) for b in bc))
    ref = po.solve(f, h, bc, zdtype=np.longdouble)
    e = rel_err(gpu_solve(f, h, bc, z_algorithm="cluster"), ref)
    assert e <= TOL, (nz, combo, e)


@pytest.mark.parametrize("h", [(1.0 / 32, 1.0 / 16, 1.0 / 1024), (1.0 / 1024, 1.0 / 1024, 1.0 / 16)],
                         ids=["small-shift", "large-shift"])
def test_cluster_conditioning(h):
    """dz << dx: pivots near -1, the chain of super-segments at its worst conditioned; dz >> dx: minors grow like
    |b|^32, the super-segment couplings 1 / q_256 underflow to zero (no coupling: correct)."""
    shape = (1024, 16, 32)
    for combo in ("PPN", "DDD"):
        bc = wl.parse_bc(combo)
        f = wl.random_normal(shape, 79, zero_mean=all(b in (0, 1) for b in bc))
        ref = po.solve(f, h, bc, zdtype=np.longdouble)
        e = rel_err(gpu_solve(f, h, bc, z_algorithm="cluster"), ref)
        assert e <= TOL, (combo, h, e)


def test_cluster_is_the_default_where_it_pays():
    """256 x 128 lines of 768 rows: PP_Z_AUTO takes the cluster kernel (two launches per singular solve: the kernel and
    the zero-mode line) and matches the oracle."""
    import torch
    import paper_1909_05423_b200 as pp
    shape, h, bc = (768, 128, 256), (1.0 / 256, 1.0 / 128, 1.0 / 768), wl.parse_bc("NNN")
    f = wl.random_normal(shape, 80, zero_mean=True)
    plan = pp.Plan(256, 128, 768, *h, bc)
    assert plan.launches_per_solve == 4 + 2
    u = plan.solve(torch.from_numpy(f).cuda()).cpu().numpy()
    plan.destroy()
    ref = po.solve(f, h, bc)
    assert rel_err(u, ref) <= TOL


def test_cluster_refused_where_it_does_not_apply():
    import paper_1909_05423_b200 as pp
    for nz, bcz in ((256, 1), (2304, 1), (1000, 2), (1024, 0)):
        plan = pp.Plan(16, 8, nz, 1.0, 1.0, 1.0, (1, 1, bcz))
        with pytest.raises(pp.PittPackError):
            plan.set_z_algorithm("cluster")
        plan.destroy()
