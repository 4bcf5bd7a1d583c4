"""N > 1 is "replicas only": every rank solves its own grid, no data-path
collective; the only cross-rank step is bench.py's max-over-ranks timing reduction and the rule
that rank 0 alone prints.  Covered here with world_size-2 gloo process groups on the CPU."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["PP_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%s" % os.environ["PP_PORT"],
                        rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank = dist.get_rank()
local_ms = [3.0, 5.0][rank]                      # rank 1 is the slow replica
ms = bench.max_over_ranks(local_ms)
value = bench.whole_job_gpoints(dist.get_world_size(), 1 << 20, ms)
dist.barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "value": value}))
dist.destroy_process_group()
"""


def test_max_over_ranks_and_whole_job_value_world2():
    port = str(free_port())
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", PP_PORT=port, PP_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (_, err) in zip(procs, outs):
        assert p.returncode == 0, err
    assert outs[1][0].strip() == ""                                  # only rank 0 prints
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["ms"] == 5.0                                          # the slowest rank decides
    assert res["value"] == pytest.approx(2 * (1 << 20) / 5e-3 / 1e9)  # both replicas' points count


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.25) == 1.25
    assert bench.whole_job_gpoints(1, 10 ** 9, 1000.0) == pytest.approx(1.0)


def test_reference_arm_only_rank0_works():
    """--impl reference under torchrun: ranks other than 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert res.returncode == 0 and res.stdout.strip() == ""
