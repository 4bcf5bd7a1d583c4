"""pittpack_b200: B200-native (sm_100a, fp64) direct Poisson solver -- the single-GPU hot path of
PittPack (arxiv 1909.05423).  The product is the C-ABI library ``libpittpack_b200.so``
(``include/pittpack_b200.h``); this package is its thin Python binding plus the seeded workload
generators (``workloads``).  The library is loaded on first use and there is no CPU fallback."""
from .binding import (  # noqa: F401
    KERNEL_NAMES, PP_BC_DIRICHLET, PP_BC_NEUMANN, PP_BC_PERIODIC, PP_NUM_KERNELS, PP_SUCCESS,
    PittPackError, Plan, lib, pp_plan_create, pp_plan_destroy, pp_plan_last_kernel_ms,
    pp_plan_set_profiling, pp_plan_workspace_bytes, pp_solve, pp_solve_host, strerror, version,
)

from .binding import pp_size_supported  # noqa: F401
from .slab import SlabPlan, VirtualRanks  # noqa: F401

__all__ = ["Plan", "SlabPlan", "VirtualRanks", "PittPackError", "lib", "version", "strerror"]
