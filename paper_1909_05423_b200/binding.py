"""Thin ctypes binding of the C ABI in include/pittpack_b200.h -- argument marshalling only;
every step of the solve runs in the CUDA kernels of libpittpack_b200.so.

The raw entry points are exported under their C names (``pp_plan_create`` ...); :class:`Plan`
wraps them for torch tensors (torch is used for device memory and streams only).

There is no CPU fallback: if the shared library is missing this module raises at first use.
"""
from __future__ import annotations

import ctypes
import os

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(PKG_DIR, "libpittpack_b200.so")

PP_BC_PERIODIC, PP_BC_NEUMANN, PP_BC_DIRICHLET = 0, 1, 2
PP_SUCCESS = 0
PP_NUM_KERNELS = 5
KERNEL_NAMES = ("x_fwd", "y_fwd", "z_solve", "y_inv", "x_inv")

EXPORTS = (
    "pp_plan_create", "pp_solve", "pp_solve_batch", "pp_solve_host", "pp_solve_host_batch", "pp_plan_destroy", "pp_plan_workspace_bytes",
    "pp_plan_set_profiling", "pp_plan_last_kernel_ms", "pp_plan_set_z_algorithm", "pp_plan_set_xy_fusion", "pp_plan_set_xy_pipeline", "pp_plan_launches_per_solve", "pp_size_supported", "pp_plan_set_null_space", "pp_fold_dirichlet", "pp_strerror", "pp_version",
    "pp_slab_plan_create", "pp_slab_plan_destroy", "pp_slab_local_elems", "pp_slab_chunk_elems", "pp_slab_set_exchange",
    "pp_slab_forward", "pp_slab_zsolve", "pp_slab_inverse",
    "pp_zsolve_static",
)
PP_STATIC_MAX_NZ = 4096
PP_ERR_STATIC_LIMIT = 6
PP_ZERO_MODE_NONE, PP_ZERO_MODE_ZERO_MEAN, PP_ZERO_MODE_PIN_PLANE0 = 0, 1, 2
PP_Z_AUTO, PP_Z_SWEEP, PP_Z_PARTITION, PP_Z_CLUSTER = 0, 1, 2, 3
PP_NULL_ZERO_MEAN, PP_NULL_PIN_PLANE0 = 0, 1

_lib = None


class PittPackError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} (status {status})")


def lib() -> ctypes.CDLL:
    """Load libpittpack_b200.so (once).  Fails loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} is missing: build it with `python -m paper_1909_05423_b200.build` "
            "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, dbl, i32 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int
    L.pp_plan_create.argtypes = [ctypes.POINTER(vp), i32, i32, i32, dbl, dbl, dbl, i32, i32, i32]
    L.pp_plan_create.restype = i32
    L.pp_solve.argtypes = [vp, vp, vp, vp]
    L.pp_solve.restype = i32
    L.pp_solve_batch.argtypes = [vp, vp, vp, i32, vp]
    L.pp_solve_batch.restype = i32
    L.pp_solve_host.argtypes = [vp, vp, vp, vp]
    L.pp_solve_host.restype = i32
    L.pp_solve_host_batch.argtypes = [vp, vp, vp, i32, vp]
    L.pp_solve_host_batch.restype = i32
    L.pp_plan_destroy.argtypes = [vp]
    L.pp_plan_destroy.restype = i32
    L.pp_plan_workspace_bytes.argtypes = [vp]
    L.pp_plan_workspace_bytes.restype = ctypes.c_size_t
    L.pp_plan_set_profiling.argtypes = [vp, i32]
    L.pp_plan_set_profiling.restype = i32
    L.pp_plan_last_kernel_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    L.pp_plan_last_kernel_ms.restype = i32
    L.pp_plan_set_z_algorithm.argtypes = [vp, i32]
    L.pp_plan_set_z_algorithm.restype = i32
    L.pp_plan_set_xy_fusion.argtypes = [vp, i32]
    L.pp_plan_set_xy_fusion.restype = i32
    L.pp_plan_set_xy_pipeline.argtypes = [vp, i32]
    L.pp_plan_set_xy_pipeline.restype = i32
    L.pp_plan_launches_per_solve.argtypes = [vp]
    L.pp_plan_launches_per_solve.restype = i32
    L.pp_size_supported.argtypes = [i32, i32, i32, i32]
    L.pp_size_supported.restype = i32
    L.pp_plan_set_null_space.argtypes = [vp, i32]
    L.pp_plan_set_null_space.restype = i32
    L.pp_fold_dirichlet.argtypes = [vp] * 9
    L.pp_fold_dirichlet.restype = i32
    L.pp_slab_plan_create.argtypes = [ctypes.POINTER(vp), i32, i32, i32, i32, i32, dbl, dbl, dbl, i32, i32, i32]
    L.pp_slab_plan_create.restype = i32
    L.pp_slab_plan_destroy.argtypes = [vp]
    L.pp_slab_plan_destroy.restype = i32
    L.pp_slab_local_elems.argtypes = [vp]
    L.pp_slab_local_elems.restype = ctypes.c_size_t
    L.pp_slab_chunk_elems.argtypes = [vp]
    L.pp_slab_chunk_elems.restype = ctypes.c_size_t
    L.pp_slab_set_exchange.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp)]
    L.pp_slab_set_exchange.restype = i32
    L.pp_slab_forward.argtypes = [vp, vp, vp, vp]
    L.pp_slab_forward.restype = i32
    L.pp_slab_zsolve.argtypes = [vp, vp, vp]
    L.pp_slab_zsolve.restype = i32
    L.pp_slab_inverse.argtypes = [vp, vp, vp]
    L.pp_slab_inverse.restype = i32
    L.pp_zsolve_static.argtypes = [vp, i32, i32, i32, i32, i32, dbl, vp, vp, vp]
    L.pp_zsolve_static.restype = i32
    L.pp_strerror.argtypes = [i32]
    L.pp_strerror.restype = ctypes.c_char_p
    L.pp_version.argtypes = []
    L.pp_version.restype = ctypes.c_char_p
    _lib = L
    return L


# ---------------------------------------------------------------- raw C-ABI calls, same names
def pp_plan_create(nx, ny, nz, dx, dy, dz, bc_x, bc_y, bc_z):
    """-> (status, handle).  handle is an integer address (0 on failure)."""
    h = ctypes.c_void_p(0)
    st = lib().pp_plan_create(ctypes.byref(h), int(nx), int(ny), int(nz), float(dx), float(dy), float(dz),
                              int(bc_x), int(bc_y), int(bc_z))
    return st, (h.value or 0)


def pp_solve(plan, f_ptr, u_ptr, stream=0):
    return lib().pp_solve(ctypes.c_void_p(plan), ctypes.c_void_p(f_ptr), ctypes.c_void_p(u_ptr),
                          ctypes.c_void_p(stream))


def pp_solve_batch(plan, f_ptr, u_ptr, nbatch, stream=0):
    return lib().pp_solve_batch(ctypes.c_void_p(plan), ctypes.c_void_p(f_ptr), ctypes.c_void_p(u_ptr), int(nbatch),
                                ctypes.c_void_p(stream))


def pp_solve_host(plan, f_ptr, u_ptr, stream=0):
    return lib().pp_solve_host(ctypes.c_void_p(plan), ctypes.c_void_p(f_ptr), ctypes.c_void_p(u_ptr),
                               ctypes.c_void_p(stream))


def pp_solve_host_batch(plan, f_ptr, u_ptr, nbatch, stream=0):
    return lib().pp_solve_host_batch(ctypes.c_void_p(plan), ctypes.c_void_p(f_ptr), ctypes.c_void_p(u_ptr), int(nbatch),
                                     ctypes.c_void_p(stream))


def pp_plan_destroy(plan):
    return lib().pp_plan_destroy(ctypes.c_void_p(plan))


def pp_plan_workspace_bytes(plan):
    return int(lib().pp_plan_workspace_bytes(ctypes.c_void_p(plan)))


def pp_plan_set_profiling(plan, enable):
    return lib().pp_plan_set_profiling(ctypes.c_void_p(plan), int(bool(enable)))


def pp_plan_last_kernel_ms(plan):
    """-> (status, [ms] * PP_NUM_KERNELS)"""
    buf = (ctypes.c_float * PP_NUM_KERNELS)()
    st = lib().pp_plan_last_kernel_ms(ctypes.c_void_p(plan), buf)
    return st, [float(v) for v in buf]


def pp_plan_set_z_algorithm(plan, algorithm):
    return lib().pp_plan_set_z_algorithm(ctypes.c_void_p(plan), int(algorithm))


def pp_plan_set_xy_fusion(plan, enable):
    return lib().pp_plan_set_xy_fusion(ctypes.c_void_p(plan), int(bool(enable)))


def pp_plan_set_xy_pipeline(plan, planes_per_slab):
    return lib().pp_plan_set_xy_pipeline(ctypes.c_void_p(plan), int(planes_per_slab))


def pp_plan_launches_per_solve(plan):
    return int(lib().pp_plan_launches_per_solve(ctypes.c_void_p(plan)))


def pp_size_supported(nx, ny, nz, bc_z):
    return bool(lib().pp_size_supported(int(nx), int(ny), int(nz), int(bc_z)))


def pp_plan_set_null_space(plan, convention):
    return lib().pp_plan_set_null_space(ctypes.c_void_p(plan), int(convention))


def pp_fold_dirichlet(plan, f_ptr, gx_lo=0, gx_hi=0, gy_lo=0, gy_hi=0, gz_lo=0, gz_hi=0, stream=0):
    """Face pointers are device addresses (0 = no face)."""
    args = [ctypes.c_void_p(int(a)) for a in (plan, f_ptr, gx_lo, gx_hi, gy_lo, gy_hi, gz_lo, gz_hi, stream)]
    return lib().pp_fold_dirichlet(*args)


def pp_slab_plan_create(world, rank, nx, ny, nz, dx, dy, dz, bc_x, bc_y, bc_z):
    """-> (status, handle)"""
    h = ctypes.c_void_p(0)
    st = lib().pp_slab_plan_create(ctypes.byref(h), int(world), int(rank), int(nx), int(ny), int(nz), float(dx), float(dy),
                                   float(dz), int(bc_x), int(bc_y), int(bc_z))
    return st, (h.value or 0)


def pp_slab_plan_destroy(plan):
    return lib().pp_slab_plan_destroy(ctypes.c_void_p(plan))


def pp_slab_local_elems(plan):
    return int(lib().pp_slab_local_elems(ctypes.c_void_p(plan)))


def pp_slab_chunk_elems(plan):
    return int(lib().pp_slab_chunk_elems(ctypes.c_void_p(plan)))


def pp_slab_set_exchange(plan, fwd_dst, inv_src):
    """fwd_dst, inv_src: sequences of `world` device addresses (the C function reads exactly `world` entries of each)."""
    n = len(fwd_dst)
    if plan:
        chunk = pp_slab_chunk_elems(plan)
        world = pp_slab_local_elems(plan) // chunk if chunk else 0
        if n != world or len(inv_src) != world:
            raise ValueError(f"pp_slab_set_exchange: need {world} addresses in fwd_dst and in inv_src, got {n} and {len(inv_src)}")
    a = (ctypes.c_void_p * n)(*[ctypes.c_void_p(int(v)) for v in fwd_dst])
    b = (ctypes.c_void_p * n)(*[ctypes.c_void_p(int(v)) for v in inv_src])
    return lib().pp_slab_set_exchange(ctypes.c_void_p(plan), a, b)


def pp_slab_forward(plan, f_ptr, work_ptr, stream=0):
    return lib().pp_slab_forward(ctypes.c_void_p(plan), ctypes.c_void_p(f_ptr), ctypes.c_void_p(work_ptr), ctypes.c_void_p(stream))


def pp_slab_zsolve(plan, pencil_ptr, stream=0):
    return lib().pp_slab_zsolve(ctypes.c_void_p(plan), ctypes.c_void_p(pencil_ptr), ctypes.c_void_p(stream))


def pp_slab_inverse(plan, u_ptr, stream=0):
    return lib().pp_slab_inverse(ctypes.c_void_p(plan), ctypes.c_void_p(u_ptr), ctypes.c_void_p(stream))


def pp_zsolve_static(w_ptr, nx, ny, nz, bc_z, zero_mode, scale, sx_ptr, sy_ptr, stream=0):
    """The plan-free z solve for callers that may not allocate device memory (see the header): w, sx, sy are
    device addresses; nz <= PP_STATIC_MAX_NZ, else PP_ERR_STATIC_LIMIT."""
    return lib().pp_zsolve_static(ctypes.c_void_p(w_ptr), int(nx), int(ny), int(nz), int(bc_z), int(zero_mode),
                                  float(scale), ctypes.c_void_p(sx_ptr), ctypes.c_void_p(sy_ptr), ctypes.c_void_p(stream))


def strerror(status: int) -> str:
    return lib().pp_strerror(int(status)).decode()


def version() -> str:
    return lib().pp_version().decode()


# ---------------------------------------------------------------- torch-facing wrapper
_BC = {"P": PP_BC_PERIODIC, "N": PP_BC_NEUMANN, "D": PP_BC_DIRICHLET}


def _bc_tuple(bc):
    if isinstance(bc, str):
        return tuple(_BC[c] for c in bc.upper())
    return tuple(int(b) for b in bc)


class Plan:
    """``Plan(nx, ny, nz, dx, dy, dz, bc)`` with ``bc`` = 'PPN' or a (bc_x, bc_y, bc_z) tuple.

    ``solve(f, u=None)`` takes contiguous float64 CUDA tensors of shape (nz, ny, nx) and runs on
    torch's current stream; ``u=None`` allocates the output, ``u is f`` solves in place."""

    def __init__(self, nx, ny, nz, dx, dy, dz, bc):
        self.shape = (int(nz), int(ny), int(nx))
        self.h = (float(dx), float(dy), float(dz))
        self.bc = _bc_tuple(bc)
        st, h = pp_plan_create(nx, ny, nz, dx, dy, dz, *self.bc)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_plan_create")
        self.handle = h
        import torch
        self.device = torch.cuda.current_device()      # the plan's tables live there (pp_plan_create)

    def _check(self, t, name):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and tuple(t.shape) == self.shape):
            raise ValueError(f"{name}: need a contiguous float64 CUDA tensor of shape {self.shape}")
        if t.device.index != self.device:
            raise ValueError(f"{name}: tensor on cuda:{t.device.index}, plan created on cuda:{self.device}")

    def solve(self, f, u=None, stream=None):
        import torch
        self._check(f, "f")
        if u is None:
            u = torch.empty_like(f)
        self._check(u, "u")
        s = torch.cuda.current_stream(f.device) if stream is None else stream
        st = pp_solve(self.handle, f.data_ptr(), u.data_ptr(), s.cuda_stream)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_solve")
        return u

    def solve_batch(self, f, u=None, stream=None):
        """f: contiguous float64 CUDA tensor (nbatch, nz, ny, nx); returns u of the same shape."""
        import torch
        if not (isinstance(f, torch.Tensor) and f.is_cuda and f.dtype == torch.float64 and f.is_contiguous()
                and f.dim() == 4 and tuple(f.shape[1:]) == self.shape):
            raise ValueError(f"f: need a contiguous float64 CUDA tensor of shape (nbatch,) + {self.shape}")
        if u is None:
            u = torch.empty_like(f)
        if not (u.is_cuda and u.dtype == torch.float64 and u.is_contiguous() and u.shape == f.shape):
            raise ValueError("u: same shape, dtype and device as f")
        if f.device.index != self.device or u.device.index != self.device:
            raise ValueError(f"tensors must live on cuda:{self.device}")
        s = torch.cuda.current_stream(f.device) if stream is None else stream
        st = pp_solve_batch(self.handle, f.data_ptr(), u.data_ptr(), f.shape[0], s.cuda_stream)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_solve_batch")
        return u

    def solve_host(self, f_host, u_host, stream=None):
        """f_host, u_host: contiguous float64 CPU tensors (pinned recommended) of the plan's shape."""
        import torch
        for t, name in ((f_host, "f_host"), (u_host, "u_host")):
            if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float64
                    and t.is_contiguous() and tuple(t.shape) == self.shape):
                raise ValueError(f"{name}: need a contiguous float64 CPU tensor of shape {self.shape}")
        s = torch.cuda.current_stream() if stream is None else stream
        st = pp_solve_host(self.handle, f_host.data_ptr(), u_host.data_ptr(), s.cuda_stream)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_solve_host")
        return u_host

    def solve_host_batch(self, f_host, u_host, stream=None):
        """f_host, u_host: contiguous float64 CPU tensors of shape (nbatch, nz, ny, nx), pinned recommended."""
        import torch
        for t, name in ((f_host, "f_host"), (u_host, "u_host")):
            if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                    and t.dim() == 4 and tuple(t.shape[1:]) == self.shape and t.shape[0] == f_host.shape[0]):
                raise ValueError(f"{name}: need a contiguous float64 CPU tensor of shape (nbatch,) + {self.shape}")
        s = torch.cuda.current_stream() if stream is None else stream
        st = pp_solve_host_batch(self.handle, f_host.data_ptr(), u_host.data_ptr(), int(f_host.shape[0]), s.cuda_stream)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_solve_host_batch")
        return u_host

    def set_profiling(self, enable: bool):
        st = pp_plan_set_profiling(self.handle, enable)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_plan_set_profiling")

    def last_kernel_ms(self):
        st, ms = pp_plan_last_kernel_ms(self.handle)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_plan_last_kernel_ms")
        return dict(zip(KERNEL_NAMES, ms))

    def set_z_algorithm(self, algorithm):
        """'auto' | 'sweep' | 'partition' (or a PP_Z_* value)."""
        alg = {"auto": PP_Z_AUTO, "sweep": PP_Z_SWEEP, "partition": PP_Z_PARTITION, "cluster": PP_Z_CLUSTER}.get(algorithm, algorithm)
        st = pp_plan_set_z_algorithm(self.handle, alg)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_plan_set_z_algorithm")

    def set_xy_fusion(self, enable: bool):
        st = pp_plan_set_xy_fusion(self.handle, enable)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_plan_set_xy_fusion")

    def set_xy_pipeline(self, planes_per_slab: int):
        st = pp_plan_set_xy_pipeline(self.handle, planes_per_slab)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_plan_set_xy_pipeline")

    def fold_dirichlet(self, f, faces, stream=None):
        """``faces``: {('x'|'y'|'z', 0|1): float64 CUDA tensor of face values}; f is modified in place."""
        import torch
        self._check(f, "f")
        nz, ny, nx = self.shape
        want = {"x": (nz, ny), "y": (nz, nx), "z": (ny, nx)}
        ptr = {}
        for (axis, side), g in faces.items():
            if not (isinstance(g, torch.Tensor) and g.is_cuda and g.dtype == torch.float64 and g.is_contiguous()
                    and tuple(g.shape) == want[axis]):
                raise ValueError(f"face {axis}{side}: need a contiguous float64 CUDA tensor of shape {want[axis]}")
            ptr[(axis, side)] = g.data_ptr()
        s = torch.cuda.current_stream(f.device) if stream is None else stream
        st = pp_fold_dirichlet(self.handle, f.data_ptr(), *(ptr.get((a, k), 0) for a in "xyz" for k in (0, 1)),
                               stream=s.cuda_stream)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_fold_dirichlet")
        return f

    def set_null_space(self, convention):
        """'zero_mean' | 'pin_plane0' (or a PP_NULL_* value)."""
        c = {"zero_mean": PP_NULL_ZERO_MEAN, "pin_plane0": PP_NULL_PIN_PLANE0}.get(convention, convention)
        st = pp_plan_set_null_space(self.handle, c)
        if st != PP_SUCCESS:
            raise PittPackError(st, "pp_plan_set_null_space")

    @property
    def launches_per_solve(self):
        return pp_plan_launches_per_solve(self.handle)

    @property
    def workspace_bytes(self):
        return pp_plan_workspace_bytes(self.handle)

    def destroy(self):
        if getattr(self, "handle", 0):
            pp_plan_destroy(self.handle)
            self.handle = 0

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
