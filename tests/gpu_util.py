"""Helpers shared by the GPU parity tests: run the CUDA path through the C ABI on a workload and
compare with the oracle.  Tolerance: north_star's max relative error <= 1e-11, measured as
max|u_gpu - u_ref| / max|u_ref| (R23)."""
import numpy as np

TOL = 1e-11


def gpu_solve(f: np.ndarray, h, bc, in_place=False, z_algorithm=None):
    import torch
    import paper_1909_05423_b200 as pp
    nz, ny, nx = f.shape
    plan = pp.Plan(nx, ny, nz, h[0], h[1], h[2], bc)
    if z_algorithm is not None:
        plan.set_z_algorithm(z_algorithm)
    ft = torch.from_numpy(np.ascontiguousarray(f)).cuda()
    ut = plan.solve(ft, ft if in_place else None)
    torch.cuda.synchronize()
    u = ut.cpu().numpy()
    plan.destroy()
    return u


def rel_err(u, ref):
    return float(np.max(np.abs(u - ref)) / max(np.max(np.abs(ref)), np.finfo(np.float64).tiny))
