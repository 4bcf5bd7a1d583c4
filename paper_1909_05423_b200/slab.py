"""Slab decomposition over several GPUs (include/pittpack_b200.h, "Slab decomposition"):
bookkeeping and plumbing only -- every arithmetic step runs in the library's kernels.

Rank r owns the z-slab ``f[r nz/P : (r+1) nz/P]`` and, for the z solve, the pencil of wavenumber rows
``ky in [r ny/P, (r+1) ny/P)`` (layout ``(nz, ny/P, nx)``).  The re-orientation between the two is fused into
the y passes, which are given the addresses of the chunks (``pp_slab_set_exchange``):

* ``SlabPlan.solve`` -- one process per GPU, ``torch.distributed`` (NCCL) all-to-all between the passes:
  the forward y pass writes a send buffer chunk by chunk, the all-to-all's receive buffer is the pencil;
  the pencil is the send buffer of the return all-to-all, the inverse y pass reads the receive buffer.
* ``VirtualRanks`` -- all ranks in ONE process on one device (their "peer" pointers are plain device
  pointers): the forward y pass of rank r stores straight into pencil q, the inverse y pass loads
  straight from it -- the peer-memory (NVLink) mode of the same kernels, which is how the multi-rank path
  is tested on a single GPU.
"""
from __future__ import annotations

from . import binding as b


def slab_extents(world: int, shape):
    """(nzl, nyl, chunk_elems) of a (nz, ny, nx) grid cut into `world` slabs / pencils."""
    nz, ny, nx = shape
    if nz % world or ny % world:
        raise ValueError(f"nz = {nz} and ny = {ny} must be multiples of world = {world}")
    nzl, nyl = nz // world, ny // world
    return nzl, nyl, nzl * nyl * nx


def chunk_offset(world: int, shape, src: int) -> int:
    """Offset (in doubles) inside ANY rank's pencil of the chunk that comes from slab `src`: the pencil is
    [nz][ny/P][nx] and slab `src` holds its planes src nz/P ... , so chunks are consecutive."""
    return src * slab_extents(world, shape)[2]


def slab_of(f, world: int, rank: int):
    """This rank's z-slab of a global (nz, ny, nx) array (a view)."""
    nzl = f.shape[0] // world
    return f[rank * nzl:(rank + 1) * nzl]


class SlabPlan:
    """One rank of the slab-decomposed solve.  ``bc`` as for :class:`binding.Plan`."""

    def __init__(self, world, rank, nx, ny, nz, dx, dy, dz, bc):
        self.world, self.rank = int(world), int(rank)
        self.shape = (int(nz), int(ny), int(nx))
        self.bc = b._bc_tuple(bc)
        self.nzl, self.nyl, self.chunk = slab_extents(self.world, self.shape)
        st, h = b.pp_slab_plan_create(world, rank, nx, ny, nz, dx, dy, dz, *self.bc)
        if st != b.PP_SUCCESS:
            raise b.PittPackError(st, "pp_slab_plan_create")
        self.handle = h
        assert b.pp_slab_local_elems(h) == self.chunk * self.world and b.pp_slab_chunk_elems(h) == self.chunk
        self._bufs = None

    # ------------------------------------------------------------------ raw phases
    def set_exchange(self, fwd_dst, inv_src):
        st = b.pp_slab_set_exchange(self.handle, list(fwd_dst), list(inv_src))
        if st != b.PP_SUCCESS:
            raise b.PittPackError(st, "pp_slab_set_exchange")

    def _stream(self, stream):
        import torch
        return (torch.cuda.current_stream() if stream is None else stream).cuda_stream

    def forward(self, f_slab, work_slab, stream=None):
        st = b.pp_slab_forward(self.handle, f_slab.data_ptr(), work_slab.data_ptr(), self._stream(stream))
        if st != b.PP_SUCCESS:
            raise b.PittPackError(st, "pp_slab_forward")

    def zsolve(self, pencil, stream=None):
        st = b.pp_slab_zsolve(self.handle, pencil.data_ptr(), self._stream(stream))
        if st != b.PP_SUCCESS:
            raise b.PittPackError(st, "pp_slab_zsolve")

    def inverse(self, u_slab, stream=None):
        st = b.pp_slab_inverse(self.handle, u_slab.data_ptr(), self._stream(stream))
        if st != b.PP_SUCCESS:
            raise b.PittPackError(st, "pp_slab_inverse")

    # ------------------------------------------------------------------ one process per GPU, NCCL all-to-all
    def solve(self, f_slab, u_slab=None, group=None):
        """Distributed solve: ``f_slab`` is this rank's (nz/P, ny, nx) slab; returns its slab of u.
        Needs an initialised ``torch.distributed`` process group of size `world` (NCCL)."""
        import torch
        import torch.distributed as dist
        if tuple(f_slab.shape) != (self.nzl,) + self.shape[1:]:
            raise ValueError(f"f_slab: need shape {(self.nzl,) + self.shape[1:]}")
        if u_slab is None:
            u_slab = torch.empty_like(f_slab)
        if self._bufs is None:
            sendrecv = torch.empty(self.world * self.chunk, dtype=torch.float64, device=f_slab.device)
            pencil = torch.empty(self.world * self.chunk, dtype=torch.float64, device=f_slab.device)
            self._bufs = (sendrecv, pencil)
            esz = 8
            chunks = [sendrecv.data_ptr() + q * self.chunk * esz for q in range(self.world)]
            self.set_exchange(chunks, chunks)       # forward writes chunk q of the buffer, inverse reads chunk q of it
        sendrecv, pencil = self._bufs
        self.forward(f_slab, u_slab)
        dist.all_to_all_single(pencil, sendrecv, group=group)        # chunk(rank -> q) lands as planes rank nz/P.. of pencil q
        self.zsolve(pencil)
        dist.all_to_all_single(sendrecv, pencil, group=group)        # chunk q of the receive buffer = rows of pencil q
        self.inverse(u_slab)
        return u_slab

    def destroy(self):
        if getattr(self, "handle", 0):
            b.pp_slab_plan_destroy(self.handle)
            self.handle = 0

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class VirtualRanks:
    """`world` ranks in one process on the current device, coupled through direct ("peer") pointers: rank r's
    forward y pass stores into pencil q at chunk r, rank r's inverse y pass loads from there."""

    def __init__(self, world, nx, ny, nz, dx, dy, dz, bc):
        import torch
        self.world = int(world)
        self.plans = [SlabPlan(world, r, nx, ny, nz, dx, dy, dz, bc) for r in range(self.world)]
        p0 = self.plans[0]
        self.pencils = [torch.empty(p0.world * p0.chunk, dtype=torch.float64, device="cuda") for _ in range(self.world)]
        for r, p in enumerate(self.plans):
            peers = [self.pencils[q].data_ptr() + r * p.chunk * 8 for q in range(self.world)]
            p.set_exchange(peers, peers)

    def solve(self, f):
        """f: global (nz, ny, nx) CUDA tensor; returns the global u assembled from the ranks' slabs."""
        import torch
        u = torch.empty_like(f)
        for r, p in enumerate(self.plans):
            p.forward(slab_of(f, self.world, r), slab_of(u, self.world, r))
        # (ranks on separate GPUs: barrier here -- every pencil complete before its z solve)
        for q, p in enumerate(self.plans):
            p.zsolve(self.pencils[q])
        # (barrier)
        for r, p in enumerate(self.plans):
            p.inverse(slab_of(u, self.world, r))
        return u

    def destroy(self):
        for p in self.plans:
            p.destroy()
