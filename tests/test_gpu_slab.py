"""Slab decomposition (the paper's pencil decomposition + all-to-all): `world`
virtual ranks on ONE device, coupled through direct pointers exactly as peers over NVLink would be -- the
forward y pass of every rank stores into the other ranks' pencils, the inverse y pass loads from them.
Element-wise parity with the oracle; and the decomposed solve must equal the single-plan solve bit for bit
(same kernels, same arithmetic, only the addresses differ)."""
import numpy as np
import pytest

from oracle import poisson_oracle as po
from paper_1909_05423_b200 import workloads as wl
from gpu_util import TOL, gpu_solve, rel_err

pytestmark = pytest.mark.gpu


def slab_solve(f, h, bc, world):
    import torch
    import paper_1909_05423_b200 as pp
    nz, ny, nx = f.shape
    vr = pp.VirtualRanks(world, nx, ny, nz, h[0], h[1], h[2], bc)
    u = vr.solve(torch.from_numpy(f).cuda())
    torch.cuda.synchronize()
    out = u.cpu().numpy()
    vr.destroy()
    return out


@pytest.mark.parametrize("world", [2, 4])
@pytest.mark.parametrize("combo", ["PPN", "NND", "DDD", "NNN", "PPP", "DPN", "NPD"])
def test_virtual_ranks_match_oracle(world, combo):
    bc = wl.parse_bc(combo)
    shape, h = (32, 64, 128), (1.0 / 128, 1.0 / 64, 1.0 / 32)          # (nz, ny, nx): all different
    f = wl.random_normal(shape, 4242 + world, zero_mean=all(b in (0, 1) for b in bc))
    ref = po.solve(f, h, bc)
    u = slab_solve(f, h, bc, world)
    assert rel_err(u, ref) <= TOL
    assert np.array_equal(u, gpu_solve(f, h, bc))                       # identical to the undecomposed solve


@pytest.mark.parametrize("shape,world", [((24, 48, 96), 2), ((12, 80, 48), 4), ((64, 16, 16), 8), ((2048, 32, 32), 4),
                                         ((100, 64, 64), 2)])
def test_virtual_ranks_other_shapes(shape, world):
    """mixed-radix lengths, ny/world = 2 rows per pencil, a two-sweep nz and a long partitioned line"""
    for combo in ("PPN", "NND"):
        bc = wl.parse_bc(combo)
        h = (0.02, 0.03, 0.025)
        f = wl.random_normal(shape, 77, zero_mean=all(b in (0, 1) for b in bc))
        u = slab_solve(f, h, bc, world)
        assert rel_err(u, po.solve(f, h, bc)) <= TOL
        assert np.array_equal(u, gpu_solve(f, h, bc))


@pytest.mark.parametrize("world", [2, 4])
def test_virtual_ranks_long_lines_follow_the_pencil(world):
    """nz = 768 on a 256 x 256 plane: the whole grid takes the cluster z kernel; a pencil of 256 x 128 lines still does,
    one of 256 x 64 lines is below the cluster rule's line count and takes the two-level partition, whose scratch the
    slab plan sizes for the pencil (it used to fall back to the two-sweep kernel: no scratch had been allocated)."""
    shape, h = (768, 256, 256), (0.02, 0.03, 0.025)
    for combo in ("NND", "NNN"):
        bc = wl.parse_bc(combo)
        f = wl.random_normal(shape, 78, zero_mean=all(b in (0, 1) for b in bc))
        u = slab_solve(f, h, bc, world)
        assert rel_err(u, po.solve(f, h, bc)) <= TOL


def test_slab_plan_argument_checks():
    import paper_1909_05423_b200 as pp
    from paper_1909_05423_b200 import binding as b
    assert b.pp_slab_plan_create(3, 0, 32, 32, 32, 0.1, 0.1, 0.1, 0, 0, 1)[0] == 2        # 32 % 3
    assert b.pp_slab_plan_create(2, 2, 32, 32, 32, 0.1, 0.1, 0.1, 0, 0, 1)[0] == 1        # rank out of range
    assert b.pp_slab_plan_create(32, 0, 32, 32, 32, 0.1, 0.1, 0.1, 0, 0, 1)[0] == 1       # world > 16
    assert b.pp_slab_plan_create(16, 0, 32, 32, 16, 0.1, 0.1, 0.1, 0, 0, 1)[0] == 2       # one plane per slab
    p = pp.SlabPlan(2, 1, 32, 32, 32, 0.1, 0.1, 0.1, "PPN")
    import torch
    x = torch.zeros(16, 32, 32, dtype=torch.float64, device="cuda")
    with pytest.raises(pp.PittPackError):
        p.forward(x, x)                                                                   # exchange addresses not set
    with pytest.raises(ValueError):
        p.set_exchange([x.data_ptr()], [x.data_ptr()])                                    # one address for world = 2
    p.destroy()


@pytest.mark.parametrize("combo", ["PPN", "NND", "NNN"])
def test_two_processes_one_gpu_peer_pointers_over_cuda_ipc(combo):
    """The multi-process form of the decomposed solve, on the one GPU there is: two processes, each with its own SlabPlan
    and its own pencil, the pencils exported to each other by CUDA IPC and used as the peer addresses of the fused y
    passes (tests/slab_ipc_worker.py).  Element-wise against the oracle."""
    import torch.multiprocessing as mp
    import slab_ipc_worker
    world, shape, h = 2, (32, 64, 128), (1.0 / 128, 1.0 / 64, 1.0 / 32)
    bc = wl.parse_bc(combo)
    f = wl.random_normal(shape, 4300, zero_mean=all(b in (0, 1) for b in bc))
    ctx = mp.get_context("spawn")
    queues = [ctx.Queue() for _ in range(world)]
    results, barrier = ctx.Queue(), ctx.Barrier(world)
    nzl = shape[0] // world
    procs = [ctx.Process(target=slab_ipc_worker.run_rank,
                         args=(r, world, (shape[2], shape[1], shape[0]), h, bc, np.ascontiguousarray(f[r * nzl:(r + 1) * nzl]),
                               queues, barrier, results)) for r in range(world)]
    for p in procs:
        p.start()
    try:
        got = {}
        for _ in range(world):
            rank, u, err = results.get(timeout=300)
            assert err is None, f"rank {rank}:\n{err}"
            got[rank] = u
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.kill()                      # exactly the process started here
    u = np.concatenate([got[r] for r in range(world)])
    assert rel_err(u, po.solve(f, h, bc)) <= TOL
    assert np.array_equal(u, gpu_solve(f, h, bc))                       # identical to the undecomposed solve
