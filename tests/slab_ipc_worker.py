"""One rank of the slab-decomposed solve as a process of its own (tests/test_gpu_slab.py, two processes on one GPU).

Each process creates its SlabPlan, allocates its own pencil, exports it to the other ranks by CUDA IPC (a CUDA tensor sent
through a multiprocessing queue travels as a cudaIpcMemHandle and is mapped on arrival) and gives the mapped addresses to
pp_slab_set_exchange: the peer-pointer mode of the fused y passes across process boundaries, which VirtualRanks (one process,
plain device pointers) does not exercise.  The three phases are separated by a cross-process barrier after a device sync --
the place an NCCL collective or a stream-ordered signal takes when the ranks sit on different GPUs."""
import traceback

WAIT = 120.0


def run_rank(rank, world, dims, h, bc, f_slab, queues, barrier, results):
    try:
        import torch
        torch.cuda.set_device(0)
        from paper_1909_05423_b200 import slab
        nx, ny, nz = dims
        plan = slab.SlabPlan(world, rank, nx, ny, nz, *h, bc)
        pencil = torch.zeros(world * plan.chunk, dtype=torch.float64, device="cuda")
        for q in range(world):
            if q != rank:
                queues[q].put((rank, pencil))                      # exported by CUDA IPC
        pencils = {rank: pencil}
        for _ in range(world - 1):
            src, t = queues[rank].get(timeout=WAIT)                # mapped into this process
            pencils[src] = t
        peers = [pencils[q].data_ptr() + rank * plan.chunk * 8 for q in range(world)]
        plan.set_exchange(peers, peers)
        f = torch.from_numpy(f_slab).cuda()
        u = torch.empty_like(f)
        plan.forward(f, u)                                         # stores chunk(rank -> q) straight into pencil q
        torch.cuda.synchronize()
        barrier.wait(WAIT)
        plan.zsolve(pencil)
        torch.cuda.synchronize()
        barrier.wait(WAIT)
        plan.inverse(u)                                            # loads chunk(rank <- q) straight from pencil q
        torch.cuda.synchronize()
        results.put((rank, u.cpu().numpy(), None))
        barrier.wait(WAIT)                                         # nobody frees a pencil a peer may still read
        plan.destroy()
    except Exception:                                              # noqa: BLE001 -- reported to the parent
        try:
            barrier.abort()
        except Exception:                                          # noqa: BLE001
            pass
        results.put((rank, None, traceback.format_exc()))
