"""Seeded synthetic inputs shaped like the paper's workloads ("Input recipe").

This module holds *no* arithmetic of the method (no transforms, no eigenvalues, no
tridiagonal solves): only source terms ``f`` on cell centres and, for manufactured
solutions, the analytic ``u`` they were derived from.  It is the one module the tests use
to feed the same arrays to the CUDA path and to the oracle; it imports neither.

The paper measures on no public data set -- only on manufactured fields and on grids sized
per GPU -- so these synthetic fields *are* the workload.

Array convention: shape ``(nz, ny, nx)``, x fastest, value at ``((i+1/2)dx, (j+1/2)dy, (k+1/2)dz)``.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

P, N, D = 0, 1, 2
BC_CHAR = {"P": P, "N": N, "D": D}
BASE_SEED = 190905423


def parse_bc(s: str):
    """'PPN' -> (0, 0, 1)   (x, y, z)."""
    return tuple(BC_CHAR[c] for c in s.upper())


def seed_for(config: int, variant: int = 0) -> int:
    return BASE_SEED + 100 * config + variant


@dataclass
class Workload:
    name: str
    shape: tuple            # (nz, ny, nx)
    h: tuple                # (dx, dy, dz)
    bc: tuple               # (bc_x, bc_y, bc_z)
    f: np.ndarray
    u_exact: np.ndarray | None = None   # analytic solution of the continuous problem, if any
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def n_points(self) -> int:
        return int(np.prod(self.shape))


def centres(n: int, h: float) -> np.ndarray:
    return (np.arange(n, dtype=np.float64) + 0.5) * h


def outer3(gz, gy, gx) -> np.ndarray:
    return gz[:, None, None] * gy[None, :, None] * gx[None, None, :]


# ------------------------------------------------------------------ random sources
def random_normal(shape, seed: int, zero_mean: bool) -> np.ndarray:
    rng = np.random.default_rng(seed)
    f = rng.standard_normal(shape)
    if zero_mean:
        f -= f.mean()
    return f


def random_uniform(shape, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.uniform(-1.0, 1.0, size=shape)


# ------------------------------------------------------------------ manufactured solutions
def mms_axis(bc: int, n: int, h: float, omega: float, phase: str | None = None):
    """1-D factor g(x) on cell centres and its frequency w (g'' = -w^2 g) compatible with the
    homogeneous boundary condition on a domain of length L = n h:
        periodic  -> cos(w x) (or sin with phase='sin'), w = 2 pi omega / L
        Neumann   -> cos(w x),                           w = pi omega / L
        Dirichlet -> sin(w x),                           w = pi omega / L
    ("Depending on the boundary conditions on each direction appropriate
    trigonometric function is selected"; R17: real functions.)"""
    L = n * h
    x = centres(n, h)
    if bc == P:
        w = 2.0 * np.pi * omega / L
        g = np.sin(w * x) if phase == "sin" else np.cos(w * x)
    elif bc == N:
        w = np.pi * omega / L
        g = np.cos(w * x)
    elif bc == D:
        w = np.pi * omega / L
        g = np.sin(w * x)
    else:
        raise ValueError(bc)
    return g, w


def mms(shape, h, bc, omega=(1, 1, 1), phase=(None, None, None)):
    """u = gx(x) gy(y) gz(z),  f = -(wx^2 + wy^2 + wz^2) u."""
    nz, ny, nx = shape
    gx, wx = mms_axis(bc[0], nx, h[0], omega[0], phase[0])
    gy, wy = mms_axis(bc[1], ny, h[1], omega[1], phase[1])
    gz, wz = mms_axis(bc[2], nz, h[2], omega[2], phase[2])
    u = outer3(gz, gy, gx)
    f = -(wx * wx + wy * wy + wz * wz) * u
    return f, u, (wx, wy, wz)


# ------------------------------------------------------------------ BASELINE.json configs
def config1(variant: str = "mms") -> Workload:
    """32^3, periodic x/y + Dirichlet z, unit cube."""
    n = 32
    shape, h, bc = (n, n, n), (1.0 / n,) * 3, (P, P, D)
    if variant == "mms":
        # u = sin(2 pi x) sin(2 pi y) sin(pi z), f = -(9 pi^2) u
        f, u, _ = mms(shape, h, bc, omega=(1, 1, 1), phase=("sin", "sin", None))
        return Workload("cfg1-32^3-PPD-mms", shape, h, bc, f, u)
    f = random_uniform(shape, seed_for(1, 0))
    return Workload("cfg1-32^3-PPD-uniform", shape, h, bc, f)


CONFIG2_COMBOS = ("DDD", "NND", "PPD", "NNN", "PPP", "PPN")   # Tables 3-7 + config 3's (R22)


def config2(combo: str, variant: str = "mms", n: int = 128) -> Workload:
    """n^3 (default 128^3), unit cube, one of the six BC combinations."""
    bc = parse_bc(combo)
    shape, h = (n, n, n), (1.0 / n,) * 3
    if variant == "mms":
        f, u, _ = mms(shape, h, bc, omega=(1, 1, 1))
        return Workload(f"cfg2-{n}^3-{combo}-mms", shape, h, bc, f, u)
    singular = all(b in (P, N) for b in bc)
    f = random_normal(shape, seed_for(2, CONFIG2_COMBOS.index(combo) if combo in CONFIG2_COMBOS else 99),
                      zero_mean=singular)
    return Workload(f"cfg2-{n}^3-{combo}-normal", shape, h, bc, f)


def config3(scale: int = 1, combo: str = "PPN") -> Workload:
    """512 x 512 x 256, periodic x/y, Neumann z, unit cube; N(0,1) projected to zero mean.
    ``scale`` > 1 divides every extent (for quick CPU-sized siblings of the headline grid); ``combo`` other
    than 'PPN' keeps grid, spacings and seed and changes the boundary conditions only (the same field,
    projected to zero mean when the combination is singular) -- for per-BC timings at the headline size."""
    nx, ny, nz = 512 // scale, 512 // scale, 256 // scale
    bc = parse_bc(combo)
    shape, h = (nz, ny, nx), (1.0 / nx, 1.0 / ny, 1.0 / nz)
    f = random_normal(shape, seed_for(3, 0), zero_mean=all(b in (P, N) for b in bc))
    return Workload(f"cfg3-{nx}x{ny}x{nz}-{combo.upper()}-normal", shape, h, bc, f)


def paper_pencil(combo: str = "PPN", nxy: int = 64, nz: int = 16384) -> Workload:
    """The paper's own per-GPU weak-scaling loads: a 64 x 64 x 16384 pencil (Fig. 8
    caption) or, with nxy = 48 and nz = 8192, the 48 x 48 x 8192 one;
    cubic cells h = 1/nxy (domain 1 x 1 x nz/nxy); N(0,1), projected to zero mean when the problem is
    singular.  Only nxy^2 tridiagonal systems, each nz long."""
    shape, h, bc = (nz, nxy, nxy), (1.0 / nxy,) * 3, parse_bc(combo)
    f = random_normal(shape, seed_for(6, 0), zero_mean=all(b in (P, N) for b in bc))
    return Workload(f"pencil-{nxy}x{nxy}x{nz}-{combo}-normal", shape, h, bc, f)


def config4(n: int = 1024, twin: bool = False) -> Workload:
    """n^3 Dirichlet x/y/z, u = sin(pi x) sin(pi y) sin(pi z).

    As written in BASELINE.json: h = 1/(n+1) (R21) -- a cell-centred grid on [0, n/(n+1)]^3, so
    the upper faces carry non-zero values g = u(face); they are folded into the source as
    PAPER.md:163 prescribes for a linearly extrapolated ghost cell: f[boundary] -= 2 g / h^2.
    ``twin=True``: h = 1/n, where the faces are homogeneous and sin(pi x) is a discrete
    eigenfunction."""
    hh = 1.0 / n if twin else 1.0 / (n + 1)
    shape, h, bc = (n, n, n), (hh,) * 3, (D, D, D)
    x = centres(n, hh)
    g = np.sin(np.pi * x)
    u = outer3(g, g, g)
    f = (-3.0 * np.pi ** 2) * u
    if not twin:
        face = n * hh                       # coordinate of the upper face on every axis
        gf = np.sin(np.pi * face)
        c = 2.0 / (hh * hh)
        f[:, :, n - 1] -= c * gf * (g[:, None] * g[None, :])     # x-face: u(face, y, z)
        f[:, n - 1, :] -= c * gf * (g[:, None] * g[None, :])     # y-face
        f[n - 1, :, :] -= c * gf * (g[:, None] * g[None, :])     # z-face
    return Workload(f"cfg4-{n}^3-DDD-{'twin' if twin else 'asgiven'}", shape, h, bc, f, u)


def config5(scale: int = 1) -> Workload:
    """2048 x 2048 x 128 anisotropic slab (dz = 4 dx), Neumann x/y, Dirichlet z; 64 Gaussian blobs."""
    nx, ny, nz = 2048 // scale, 2048 // scale, 128 // scale
    dx, dy = 1.0 / nx, 1.0 / ny
    dz = 4.0 * dx
    shape, h, bc = (nz, ny, nx), (dx, dy, dz), (N, N, D)
    rng = np.random.default_rng(seed_for(5, 0))
    nb = 64
    Lx, Ly, Lz = nx * dx, ny * dy, nz * dz
    cx, cy, cz = rng.uniform(0, Lx, nb), rng.uniform(0, Ly, nb), rng.uniform(0, Lz, nb)
    sig = rng.uniform(0.01, 0.1, nb)
    amp = rng.uniform(-1.0, 1.0, nb)
    x, y, z = centres(nx, dx), centres(ny, dy), centres(nz, dz)
    gx = np.exp(-0.5 * ((x[None, :] - cx[:, None]) / sig[:, None]) ** 2)      # (nb, nx)
    gy = np.exp(-0.5 * ((y[None, :] - cy[:, None]) / sig[:, None]) ** 2)
    gz = np.exp(-0.5 * ((z[None, :] - cz[:, None]) / sig[:, None]) ** 2) * amp[:, None]
    f = np.empty(shape)
    for k in range(nz):                     # one plane at a time keeps the temporaries small
        f[k] = (gy * gz[:, k][:, None]).T @ gx
    return Workload(f"cfg5-{nx}x{ny}x{nz}-NND-blobs", shape, h, bc, f)
