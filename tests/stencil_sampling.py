"""Sampled cells and their six neighbours for residual checks at sizes where only sampled outputs can be
compared (tests/test_gpu_fullsize.py) -- plain NumPy index arithmetic, shared by the CPU pin of
``oracle.stencil_at`` (tests/test_oracle_stencil.py) and the GPU tests, where torch only does the gather.

Ghost rules of the three homogeneous boundary conditions on a cell-centred grid (
``oracle.poisson_oracle.lap1d``): periodic -> wrap around, Neumann -> the cell itself (mirror),
Dirichlet -> minus the cell itself (linear extrapolation through a zero face value)."""
import numpy as np

P, N, D = 0, 1, 2


def sample_indices(shape, count, seed):
    """(k, j, i) of `count` cells: random ones, with a third of them forced onto the faces of each axis
    in turn (overlapping ranges put some on edges and corners)."""
    rng = np.random.default_rng(seed)
    nz, ny, nx = shape
    k = rng.integers(0, nz, count)
    j = rng.integers(0, ny, count)
    i = rng.integers(0, nx, count)
    third = count // 3
    k[:third] = rng.choice([0, nz - 1], third)
    j[third // 2: third + third // 2] = rng.choice([0, ny - 1], third)
    i[third: 2 * third] = rng.choice([0, nx - 1], third)
    return k, j, i


def neighbour_table(idx, shape, bc):
    """For the cells `idx` = (k, j, i): a list of seven ((kk, jj, ii), sign) entries in the column order
    of ``oracle.stencil_at`` -- centre, x-1, x+1, y-1, y+1, z-1, z+1 -- where (kk, jj, ii) are in-range cell
    indices and `sign` (+1 / -1 float array) carries the Dirichlet ghost's sign."""
    k, j, i = (np.asarray(v, dtype=np.int64) for v in idx)
    nz, ny, nx = shape
    ones = np.ones(k.shape, dtype=np.float64)
    table = [((k, j, i), ones)]
    for axis, (n, b) in enumerate(zip((nx, ny, nz), bc)):
        for d in (-1, 1):
            t = (i, j, k)[axis] + d
            outside = (t < 0) | (t >= n)
            sign = ones
            if b == P:
                t = t % n
            elif b in (N, D):
                t = np.clip(t, 0, n - 1)
                if b == D:
                    sign = np.where(outside, -1.0, 1.0)
            else:
                raise ValueError(b)
            cell = [k, j, i]
            cell[2 - axis] = t
            table.append((tuple(cell), sign))
    return table


def gather_numpy(u, table):
    """(count, 7) neighbour array from a NumPy field u[k, j, i]."""
    return np.stack([sign * u[cell] for cell, sign in table], axis=1)


def gather_torch(u, table):
    """The same gather from a CUDA tensor; returns a NumPy (count, 7) array."""
    import torch
    cols = []
    for (kk, jj, ii), sign in table:
        kk, jj, ii = (torch.from_numpy(v).to(u.device) for v in (kk, jj, ii))
        cols.append(torch.from_numpy(sign).to(u.device) * u[kk, jj, ii])
    return torch.stack(cols, dim=1).cpu().numpy()
