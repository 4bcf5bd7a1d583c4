#!/usr/bin/env python
"""Benchmark of the direct Poisson solve (BASELINE.json metric: Gpoints/s per fp64 Poisson solve and
% of HBM roofline at 512x512x256).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--workload cfg3|cfg1|cfg2|cfg4|cfg5|pencil|pencil48] [--bc PPN] [--fusion] [--no-cpu-baseline]

A "step" is one pp_solve: the whole hot path (x-fwd, y-fwd, z-solve, y-inv, x-inv) over one synthetic
grid.  N > 1 runs N independent replicas (one process per GPU, no data-path collective -- DESIGN.md
"replicas only"); value = points solved by all ranks / max-over-ranks device time.  `e2e` is the same
metric through the host-buffer entry point (pp_solve_host_batch: every step's H2D and D2H inside the
timed region, copies of neighbouring steps pipelined with the solves); `roofline` is the slowest pass
against the measured HBM copy bandwidth, `roofline_solve` the whole solve against 80 B/point.

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for the definition of every field.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Gpoints/s per fp64 Poisson solve"
UNIT = "Gpoints/s"
BYTES_PER_POINT_SOLVE = 80.0     # 5 passes x (8 B read + 8 B write)
BYTES_PER_POINT_KERNEL = 16.0    # one pass
FALLBACK_HBM_GBS = 6650.0        # /opt/skills/guides/B200_PROFILING.md


def workload_by_name(name, bc=None):
    from paper_1909_05423_b200 import workloads as wl
    if bc and name not in ("cfg3", "pencil", "pencil48"):
        raise SystemExit("--bc applies to the cfg3 grid and the pencils only")
    if name == "cfg3":
        return wl.config3(combo=bc or "PPN")
    if name == "cfg4":
        return wl.config4()
    if name == "cfg5":
        return wl.config5()
    if name == "cfg2":
        return wl.config2("PPN", "normal")
    if name == "cfg1":
        return wl.config1("uniform")
    if name == "pencil":
        return wl.paper_pencil(bc or "PPN")
    if name == "pencil48":
        return wl.paper_pencil(bc or "PPN", nxy=48, nz=8192)
    raise SystemExit(f"unknown workload {name}")


def describe(w):
    nz, ny, nx = w.shape
    bc = "".join("PND"[b] for b in w.bc)
    return f"{nx}x{ny}x{nz} fp64, bc(x,y,z)={bc}, {w.name}"


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def committed_traffic(workload, kernel):
    """dram bytes per launch of pass `kernel` at `workload` from a committed ncu --set full summary
    (profiles/dram_traffic.csv: workload,kernel,bytes,source), or None when no capture of that workload
    and kernel is committed."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    try:
        with open(path) as fh:
            for line in fh:
                t = [s.strip() for s in line.split(",")]
                if len(t) >= 3 and t[0] == workload and t[1] == kernel:
                    return float(t[2])
    except Exception:
        pass
    return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML (about every millisecond) while the
    measured regions run; a region is the slice of samples between two mark() calls."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, index, period=0.001):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.stop_flag = threading.Event()
        self.mhz, self.masks, self.max_mhz, self.ok = [], [], None, False

    def run(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            try:
                pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)
                reasons = pynvml.nvmlDeviceGetCurrentClocksEventReasons
            except Exception:
                reasons = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
            self.ok = True
            while not self.stop_flag.is_set():
                mhz = int(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                mask = int(reasons(h))
                self.masks.append(mask)
                self.mhz.append(mhz)                     # appended last: len(mhz) <= len(masks)
                time.sleep(self.period)
        except Exception as exc:  # pragma: no cover
            self.error = repr(exc)

    def mark(self):
        return len(self.mhz)

    def result(self, lo=0, hi=None):
        mhz = self.mhz[lo:hi]
        if not self.ok or not mhz:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"], "samples": 0}
        mask = 0
        for m in self.masks[lo:(lo + len(mhz))]:
            mask |= m
        s = sorted(mhz)
        return {"sm_mhz": s[len(s) // 2], "sm_min_mhz": s[0], "sm_max_mhz": self.max_mhz,
                "reasons": sorted(name for bit, name in self.REASONS.items() if mask & bit), "samples": len(s)}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ------------------------------------------------------------------------------------------
# the oracle arm (cpu_baseline and --impl reference)
# ------------------------------------------------------------------------------------------
def oracle_sample(w, step_seconds=18.0):
    """Times the oracle, as it stands, on a bounded sample of workload `w`: the full x-y extent and
    all boundary conditions, with as many z planes as fit the budget (per-point cost of the oracle is
    flat in nz: the transforms are per plane, Thomas is O(nz) per mode)."""
    import numpy as np
    from oracle import poisson_oracle as po
    nz, ny, nx = w.shape
    def probe(n):
        f = np.ascontiguousarray(w.f[:n])
        t0 = time.perf_counter()
        po.solve(f, w.h, w.bc)
        return time.perf_counter() - t0

    n1, n2 = min(nz, 2), min(nz, 10)
    probe(n1)                                     # first call pays the BLAS start-up
    t1, t2 = probe(n1), probe(n2)
    per_plane = max((t2 - t1) / max(n2 - n1, 1), 1e-6)
    fixed = max(t1 - per_plane * n1, 0.0)
    target_nz = int(max(2, min(nz, (step_seconds - fixed) / per_plane)))
    sample = {"nz": target_nz, "ny": ny, "nx": nx,
              "text": (f"oracle.poisson_oracle.solve on the first {target_nz} of {nz} z-planes of the workload "
                       f"({nx}x{ny}x{target_nz}, same spacings and BCs), one solve")}
    return sample


def time_oracle(w, sample):
    import numpy as np
    from oracle import poisson_oracle as po
    f = np.ascontiguousarray(w.f[: sample["nz"]])
    t0 = time.perf_counter()
    po.solve(f, w.h, w.bc)
    dt = time.perf_counter() - t0
    return f.size / dt / 1e9, dt


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [int(i.get("num_threads", 1)) for i in threadpool_info() if i.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return len(os.sched_getaffinity(0))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = workload_by_name(args.workload, args.bc)
    sample = oracle_sample(w, step_seconds=150.0 / max(1, args.steps + args.warmup))
    for _ in range(args.warmup):
        time_oracle(w, sample)
    vals, secs = [], []
    for _ in range(args.steps):
        v, dt = time_oracle(w, sample)
        vals.append(v)
        secs.append(dt)
    total_pts = sample["nz"] * sample["ny"] * sample["nx"] * args.steps
    value = total_pts / sum(secs) / 1e9
    cores = blas_threads()
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe(w), "sample": sample["text"]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample["text"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))
    return 0


# ------------------------------------------------------------------------------------------
# N > 1: replicas only -- the only cross-rank step is the timing reduction
# ------------------------------------------------------------------------------------------
def max_over_ranks(ms: float, device="cpu") -> float:
    """Slowest rank's device time.  Uses the default process group if one is initialised (NCCL on
    the GPU box, gloo in the CPU tests); a single process returns its own time."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gpoints(world: int, npts_per_rank: int, ms_step: float) -> float:
    """Every rank solves its own grid (weak scaling): points solved by all ranks / slowest rank's time."""
    return world * npts_per_rank / (ms_step * 1e-3) / 1e9


# ------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------
def sampled_residual(u, f, h, bc, count=200_000, seed=11):
    """max |A u - f| over `count` random cells of the timed solve's output, relative to max |f| -- eq. 3
     with the ghost rules of the three boundary conditions, by torch gathers on the device.
    (bench.py's own check that the timed kernels solved the problem; the oracle is not involved.)"""
    import torch
    nz, ny, nx = u.shape
    g = torch.Generator(device="cpu").manual_seed(seed)
    idx = [torch.randint(0, n, (count,), generator=g).to(u.device) for n in (nz, ny, nx)]
    uc = u[idx[0], idx[1], idx[2]]
    fs = f[idx[0], idx[1], idx[2]]
    if all(b in (0, 1) for b in bc):
        fs = fs - f.mean()                              # singular: the solve projects f to zero mean
    acc = torch.zeros_like(uc)
    for axis, (n, b, hh) in enumerate(zip((nx, ny, nz), bc, h)):
        for d in (-1, 1):
            cell = list(idx)
            t = cell[2 - axis] + d
            outside = (t < 0) | (t >= n)
            if b == 0:
                t = t % n
                sign = 1.0
            else:
                t = t.clamp(0, n - 1)
                sign = torch.where(outside, -1.0, 1.0) if b == 2 else 1.0
            cell[2 - axis] = t
            acc += (sign * u[cell[0], cell[1], cell[2]] - uc) / (hh * hh)
    return float((acc - fs).abs().max() / f.abs().max())


def run_cuda(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_1909_05423_b200 as pp

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus} but WORLD_SIZE={world}: launch one rank per GPU "
                         "(python -m torch.distributed.run --nproc-per-node N bench.py --gpus N ...)")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local_rank)
    distributed = world > 1
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    w = workload_by_name(args.workload, args.bc)
    nz, ny, nx = w.shape
    npts = w.n_points
    plan = pp.Plan(nx, ny, nz, *w.h, w.bc)
    if args.fusion:
        plan.set_xy_fusion(True)
    if args.xy_pipeline:
        plan.set_xy_pipeline(args.xy_pipeline)
    paired = bool(args.fusion or args.xy_pipeline)          # the x and y pass of a plane are timed as one slot
    launches = plan.launches_per_solve
    f = torch.from_numpy(w.f).cuda()
    u = torch.empty_like(f)
    stream = torch.cuda.current_stream()

    for _ in range(max(args.warmup, 3)):
        plan.solve(f, u)
    barrier()

    # ---- timed region: K solves, inputs resident in HBM (f, u: 2 x N x 8 B, far larger than L2)
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    t_wait = time.perf_counter()                        # NVML start-up can take longer than a short timed region:
    while sampler.mark() < 3 and not getattr(sampler, "error", None) and time.perf_counter() - t_wait < 10.0:
        time.sleep(0.005)                               # wait for the first samples, not for a fixed time
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    m0 = sampler.mark()
    e0.record(stream)
    for _ in range(args.steps):
        plan.solve(f, u)
    e1.record(stream)
    barrier()
    m1 = sampler.mark()
    ms_total = max_over_ranks(e0.elapsed_time(e1), "cuda")
    ms_step = ms_total / args.steps
    value = whole_job_gpoints(world, npts, ms_step)
    residual = sampled_residual(u, f, w.h, w.bc)        # of the last timed solve's output

    # ---- launch-bound grids (configs 1 and 2): the same K solves replayed from one CUDA graph
    graph_ms = None
    if npts <= (1 << 22) and world == 1:
        gs = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(gs):
            plan.solve(f, u, stream=gs)
            gs.synchronize()
            with torch.cuda.graph(graph, stream=gs):
                for _ in range(args.steps):
                    plan.solve(f, u, stream=gs)
            graph.replay()
            gs.synchronize()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(gs)
            graph.replay()
            g1.record(gs)
            gs.synchronize()
        graph_ms = g0.elapsed_time(g1) / args.steps
        del graph

    # ---- many right-hand sides as one stack (pp_solve_batch): the launch-bound grids at the large grids' speed
    batch = None
    if args.batch > 1 and world == 1:
        fb = f.unsqueeze(0).repeat(args.batch, 1, 1, 1).contiguous()
        ub = torch.empty_like(fb)
        for _ in range(3):
            plan.solve_batch(fb, ub)
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        b0.record(stream)
        for _ in range(args.steps):
            plan.solve_batch(fb, ub)
        b1.record(stream)
        torch.cuda.synchronize()
        bms = b0.elapsed_time(b1) / args.steps
        batch = {"api": "pp_solve_batch", "right_hand_sides": args.batch, "ms_per_batch": bms,
                 "value": args.batch * npts / (bms * 1e-3) / 1e9, "unit": UNIT,
                 "one_by_one_ms": ms_step * args.batch, "bit_identical_to_single_solves": bool(torch.equal(ub[args.batch - 1], u))}
        del fb, ub

    # ---- per-kernel durations over the same number of steps (CUDA events on the launching stream)
    plan.set_profiling(True)
    sums = dict.fromkeys(pp.KERNEL_NAMES, 0.0)
    barrier()
    m2 = sampler.mark()
    for _ in range(args.steps):
        plan.solve(f, u)
        for k, v in plan.last_kernel_ms().items():
            sums[k] += v
    m3 = sampler.mark()
    plan.set_profiling(False)
    kernel_ms = {k: v / args.steps for k, v in sums.items()}

    # ---- end to end through the host-buffer entry points (pinned host memory; H2D + solve + D2H of every step
    # inside the timed region): one call per step (pp_solve_host), and a pipelined batch (pp_solve_host_batch),
    # where the copy-in of step i+1 and the copy-out of step i-1 run beside the solve of step i
    e2e_steps = max(3, min(args.steps, 10))
    if args.no_e2e:
        sampler.stop_flag.set()
        sampler.join()
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "ms_per_step": ms_step, "kernel_ms": kernel_ms,
                              "config": {"workload": describe(w)}, "note": "--no-e2e: profiling run, not a bench line"}))
        plan.destroy()
        if distributed:
            dist.barrier()
            dist.destroy_process_group()
        return 0
    fh = torch.from_numpy(w.f).pin_memory()
    uh = torch.empty_like(fh).pin_memory()
    plan.solve_host(fh, uh)
    barrier()
    m4 = sampler.mark()
    e0.record(stream)
    for _ in range(e2e_steps):
        plan.solve_host(fh, uh)
    e1.record(stream)
    barrier()
    e2e_single_ms = max_over_ranks(e0.elapsed_time(e1), "cuda") / e2e_steps
    nbatch = int(min(12, (6 << 30) // (npts * 8)))              # at most 6 GiB of pinned input (and as much output) per rank: the
                                                                 # pipeline fills and drains once per call (one step's worth of copies)
    e2e_ms, e2e_api = e2e_single_ms, "pp_solve_host (pinned host buffers, one call per step)"
    if nbatch >= 3:
        fb = fh.unsqueeze(0).repeat(nbatch, 1, 1, 1).pin_memory()
        ub = torch.empty_like(fb).pin_memory()
        plan.solve_host_batch(fb, ub)                            # warm-up: allocates the staging ring
        barrier()
        t0 = time.perf_counter()                                 # the call synchronises: host clock around it
        plan.solve_host_batch(fb, ub)
        e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3 / nbatch, "cuda")
        e2e_api = f"pp_solve_host_batch (pinned host buffers, {nbatch} steps per call, copies pipelined with the solves)"
        e2e_steps = nbatch
        del fb, ub
    m5 = sampler.mark()
    sampler.stop_flag.set()
    sampler.join()
    e2e_value = whole_job_gpoints(world, npts, e2e_ms)

    if rank == 0:
        peak, peak_src = measured_peak()
        # algorithmic bytes per point of each timed slot: 16 per pass, whatever
        # the number of kernels a slot holds ("so that adding passes cannot inflate it"); with x+y fusion the pair's
        # 32 sit in the x slot.  What the kernels of a slot actually move is reported beside it: the two-level z solve
        # of long lines reads its right-hand sides twice (24 B per point).
        slot_bytes = dict.fromkeys(pp.KERNEL_NAMES, BYTES_PER_POINT_KERNEL)
        if paired:
            slot_bytes.update(x_fwd=32.0, y_fwd=0.0, y_inv=0.0, x_inv=32.0)
        xy_launches = 2 if args.fusion else (4 * -(-nz // args.xy_pipeline) if 0 < args.xy_pipeline < nz else 4)
        moved_bytes = dict(slot_bytes)
        if launches - xy_launches > 2:
            moved_bytes["z_solve"] = 24.0
        dom = max((k for k in kernel_ms if slot_bytes[k] > 0), key=lambda k: kernel_ms[k] / slot_bytes[k])
        achieved = slot_bytes[dom] * npts / (kernel_ms[dom] * 1e-3) / 1e9
        solve_gbs = BYTES_PER_POINT_SOLVE * npts / (ms_step * 1e-3) / 1e9
        wkey = (args.workload + (("-" + args.bc.upper()) if args.bc else "") + ("-fused" if args.fusion else "")
                + ("-pipelined" if args.xy_pipeline else ""))
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": describe(w), "parallelism": f"replicas x{world} (no collective)",
                       "l2_policy": "inputs larger than L2 (f and u are %d MiB each)" % (npts * 8 >> 20),
                       "in_place": False, "library": args.lib or "default build", "xy_fusion": bool(args.fusion), "xy_pipeline_planes": int(args.xy_pipeline),
                       "kernels_per_solve": launches},
            "clocks": sampler.result(m0, m1),
            "clocks_regions": {"per_kernel_timing": sampler.result(m2, m3), "e2e": sampler.result(m4, m5)},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": npts * 8, "d2h_bytes_per_step": npts * 8,
                    "ms_per_step": e2e_ms, "steps": e2e_steps, "api": e2e_api,
                    "single_call": {"value": whole_job_gpoints(world, npts, e2e_single_ms), "ms_per_step": e2e_single_ms,
                                    "api": "pp_solve_host"}},
            "gpu_launches": launches * args.steps,
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": committed_traffic(wkey, dom), "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": slot_bytes[dom] * npts,
                         "algorithmic_bytes_per_point": slot_bytes[dom], "bytes_moved_per_point": moved_bytes[dom]},
            "roofline_solve": {"bound": "hbm", "achieved": solve_gbs, "peak": peak, "unit": "GB/s",
                               "frac": solve_gbs / peak, "bytes_per_point": BYTES_PER_POINT_SOLVE,
                               "frac_of_nominal_8TBs": solve_gbs / 8000.0},
            "kernel_ms": kernel_ms,
            "kernel_gbs": {k: slot_bytes[k] * npts / (v * 1e-3) / 1e9 for k, v in kernel_ms.items() if slot_bytes[k] > 0},
            "graph_replay_ms_per_step": graph_ms,
            "batch": batch,
            "check": {"sampled_residual_rel": residual,
                      "what": "max|A u - f| / max|f| at 200000 random cells of the last timed solve's output (eq. 3)"},
        }
        if world == 1 and not args.no_cpu_baseline:
            # the oracle on a bounded sample of the workload (its first K z planes), and -- the same sample through
            # the CUDA path -- the parity error that goes with this timing
            sample = oracle_sample(w, step_seconds=18.0)
            fs = np.ascontiguousarray(w.f[: sample["nz"]])
            t0 = time.perf_counter()
            from oracle import poisson_oracle as po
            ref = po.solve(fs, w.h, w.bc)
            dt = time.perf_counter() - t0
            out["cpu_baseline"] = {"value": fs.size / dt / 1e9, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                                   "sample": sample["text"], "seconds": dt}
            if pp.pp_size_supported(nx, ny, sample["nz"], w.bc[2]):
                p2 = pp.Plan(nx, ny, sample["nz"], *w.h, w.bc)
                us = p2.solve(torch.from_numpy(fs).cuda()).cpu().numpy()
                p2.destroy()
                out["cpu_baseline"]["parity_max_rel_err"] = float(np.max(np.abs(us - ref)) / np.max(np.abs(ref)))
        print(json.dumps(out))
    plan.destroy()
    if distributed:
        dist.barrier()
        dist.destroy_process_group()
    return 0



def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start one rank per GPU ourselves (the driver's own
    multi-GPU command is the same torch.distributed.run line)."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "pencil", "pencil48"])
    ap.add_argument("--bc", default=None, help="boundary conditions (x, y, z) of the cfg3 grid or a pencil, e.g. NNN; default PPN")
    ap.add_argument("--fusion", action="store_true", help="plane-wise x+y fusion through L2 (opt-in, DESIGN.md)")
    ap.add_argument("--xy-pipeline", type=int, default=0, metavar="PLANES",
                    help="x and y passes slab by slab on two streams, PLANES planes per slab (opt-in, DESIGN.md)")
    ap.add_argument("--lib", default=None, metavar="PATH",
                    help="load this build of the library instead of the default one (a variant built with "
                         "`python -m paper_1909_05423_b200.build -D... -o PATH`: tuning switches of the kernels)")
    ap.add_argument("--batch", type=int, default=0, metavar="NB",
                    help="also time pp_solve_batch on NB copies of the workload's right-hand side (adds a `batch` key)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer (e2e) legs: for runs under a profiler")
    args = ap.parse_args()
    if args.bc is not None and (len(args.bc) != 3 or any(c not in "PNDpnd" for c in args.bc)):
        raise SystemExit("--bc: three letters out of P, N, D")
    if args.lib:
        import paper_1909_05423_b200.binding as binding
        binding.LIB_PATH = os.path.abspath(args.lib)
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
