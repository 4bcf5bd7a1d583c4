"""Rank / offset bookkeeping of the slab decomposition (paper_1909_05423_b200/slab.py) with a world_size-2 and a
world_size-4 gloo process group on the CPU: the layout identities the fused exchange relies on --
  * chunk q of rank r's send buffer, laid out [nz/P][ny/P][nx], delivered by all_to_all_single, makes the receive
    buffer of rank q exactly its pencil [nz][ny/P][nx];
  * the pencil is itself the send buffer of the return all-to-all, and block q of rank r's receive buffer holds rows
    [q ny/P, (q+1) ny/P) of its slab.
The transforms are replaced by the identity (every rank just moves the global array's entries), so a wrong offset or a
transposed extent shows up as a mismatch with the global array."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["PP_ROOT"])
import numpy as np, torch, torch.distributed as dist
from paper_1909_05423_b200.slab import slab_extents, chunk_offset, slab_of
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%s" % os.environ["PP_PORT"],
                        rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
P, r = dist.get_world_size(), dist.get_rank()
shape = (8, 12, 6)                                    # (nz, ny, nx)
nz, ny, nx = shape
G = torch.arange(nz * ny * nx, dtype=torch.float64).reshape(shape)        # the "spectrum", known to every rank
nzl, nyl, chunk = slab_extents(P, shape)
assert (nzl, nyl, chunk) == (nz // P, ny // P, nz * ny * nx // P // P)
mine = slab_of(G, P, r)                               # (nzl, ny, nx)
# what the forward y pass does with its stores: row j of local plane z -> chunk j // nyl, [z][j % nyl][:]
send = torch.empty(P * chunk, dtype=torch.float64)
for q in range(P):
    send[q * chunk:(q + 1) * chunk] = mine[:, q * nyl:(q + 1) * nyl, :].reshape(-1)
pencil = torch.empty(P * chunk, dtype=torch.float64)
dist.all_to_all_single(pencil, send)
want = G[:, r * nyl:(r + 1) * nyl, :]                 # (nz, nyl, nx): every plane, my wavenumber rows
assert torch.equal(pencil.reshape(nz, nyl, nx), want), "forward exchange"
for src in range(P):                                  # chunk_offset: where slab src's planes start inside a pencil
    o = chunk_offset(P, shape, src)
    assert torch.equal(pencil[o:o + chunk].reshape(nzl, nyl, nx), want[src * nzl:(src + 1) * nzl])
# return leg: the pencil is the send buffer; the inverse y pass reads row j of plane z from block j // nyl
recv = torch.empty(P * chunk, dtype=torch.float64)
dist.all_to_all_single(recv, pencil)
back = torch.empty_like(mine)
for q in range(P):
    back[:, q * nyl:(q + 1) * nyl, :] = recv[q * chunk:(q + 1) * chunk].reshape(nzl, nyl, nx)
assert torch.equal(back, mine), "return exchange"
dist.barrier()
dist.destroy_process_group()
print("ok", r)
"""


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 4])
def test_exchange_layout_identities(world):
    port = str(free_port())
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE=str(world), PP_PORT=port, PP_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    for rank, (p, (out, err)) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, err
        assert out.strip() == f"ok {rank}"


def test_extents_reject_indivisible_grids():
    sys.path.insert(0, ROOT)
    from paper_1909_05423_b200.slab import slab_extents
    with pytest.raises(ValueError):
        slab_extents(3, (8, 12, 6))
    assert slab_extents(4, (8, 12, 6)) == (2, 3, 36)
