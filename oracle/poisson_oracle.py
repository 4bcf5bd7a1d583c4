"""Plain, slow, obviously-correct CPU oracle of the PittPack direct Poisson solve.

TEST INFRASTRUCTURE ONLY (see ``oracle/__init__.py``).  fp64 NumPy throughout; the z
solve can optionally run in ``numpy.longdouble`` (``zdtype``) to serve as ground truth
where fp64 Thomas itself is the limiting error ("precision hazards").

What is computed (eq. 3-4):  ``u = A^-1 f`` (or ``u = A^+ f`` with ``f``
projected to zero mean when ``A`` is singular), ``A`` the 7-point second-order operator
on a cell-centred uniform grid with homogeneous periodic / Neumann / Dirichlet
conditions at the cell faces.

How (§2.1, 93-206 §3, 208-218 §4, 511-533 §7), in the paper's order:
  1. forward transform along x, then y, chosen per axis by its boundary condition
     (Table 1) -- here the *definitions* eq. 6 / 7 / 9 as naive sums
     (a dense matrix product per axis; the matmul is the only library step);
  2. for every (kx, ky) one tridiagonal system in z whose diagonal carries the summed
     modified wavenumbers of Table 2, solved by the textbook Thomas
     recurrence of Algorithm 1; periodic z by Sherman-Morrison, "two
     solves"; the singular (0,0) system by the pin / mean fix;
  3. inverse transforms along y, then x (eq. 8 / 10 as the exact inverses).

Array convention: ``f[k, j, i]`` = value at cell centre ``((i+1/2)dx, (j+1/2)dy, (k+1/2)dz)``,
shape ``(nz, ny, nx)``, x fastest.

Readings of garbled / ambiguous passages are listed in DESIGN.md ("Readings"); each is
referenced below as R<n>.
"""
from __future__ import annotations

import numpy as np

PERIODIC, NEUMANN, DIRICHLET = 0, 1, 2
BC_NAMES = {PERIODIC: "P", NEUMANN: "N", DIRICHLET: "D"}


# --------------------------------------------------------------------------------------
# 1-D building blocks
# --------------------------------------------------------------------------------------
def lap1d(n: int, bc: int) -> np.ndarray:
    """Dense 1-D second-difference matrix ``L`` (without 1/h^2) for one axis.

    PAPER.md:64 (eq. 3): interior rows (1, -2, 1).  Boundary rows after eliminating the
    ghost cell (cell-centred grid, condition imposed at the cell *face*):
      periodic  -- wrap-around neighbours;
      Neumann   -- ghost = mirror  (u_-1 = u_0)            -> corner diagonal -1;
      Dirichlet -- ghost by linear extrapolation through the face value g=0
                   (u_-1 = 2g - u_0)          -> corner diagonal -3.
    """
    L = np.zeros((n, n))
    for i in range(n):
        L[i, i] = -2.0
        if i > 0:
            L[i, i - 1] = 1.0
        if i < n - 1:
            L[i, i + 1] = 1.0
    if bc == PERIODIC:
        L[0, n - 1] += 1.0
        L[n - 1, 0] += 1.0
    elif bc == NEUMANN:
        L[0, 0] += 1.0
        L[n - 1, n - 1] += 1.0
    elif bc == DIRICHLET:
        L[0, 0] -= 1.0
        L[n - 1, n - 1] -= 1.0
    else:
        raise ValueError(f"unknown boundary condition {bc}")
    return L


def _table2(theta):
    """Table 2: ``lam = -2 + 2 cos(theta)``, evaluated as the identical ``-4 sin^2(theta / 2)``.

    The printed form cancels for small theta: at n = 2048 the lowest modes have ``1 - cos(theta) ~ 1e-6`` and
    ``-2 + 2 cos`` in fp64 keeps only ten digits of them -- the eigenvalue the whole solve divides by (reading R27,
    DESIGN.md; pinned against an 80-bit evaluation of the printed form in tests/test_oracle_operators.py)."""
    sh = np.sin(0.5 * theta)
    return -4.0 * sh * sh


def basis(n: int, bc: int):
    """Eigenbasis of ``lap1d(n, bc)``: ``(Phi, w, lam)``.

    ``Phi[i, k] = phi_k(i)``, ``w[k] = sum_i |phi_k(i)|^2``, ``lam[k]`` = Table 2
    (R8: k = 0..n-1, the 1/h^2 is applied by the caller).

      periodic   phi_k(i) = exp(+2 pi sqrt(-1) k i / n)            eq. 6,
      Neumann    phi_k(i) = cos((i + 1/2) k pi / n)                eq. 7,
      Dirichlet  phi_k(i) = sin((i + 1/2) (k + 1) pi / n)          eq. 9,

    Trigonometric arguments are reduced in integer arithmetic first (k*i mod n, resp.
    (2i+1)k mod 4n) so that large products do not lose bits in the argument.
    """
    i = np.arange(n, dtype=np.int64)[:, None]
    k = np.arange(n, dtype=np.int64)[None, :]
    kk = np.arange(n, dtype=np.float64)
    if bc == PERIODIC:
        m = (k * i) % n
        ang = 2.0 * np.pi * m.astype(np.float64) / n
        Phi = np.cos(ang) + 1j * np.sin(ang)
        w = np.full(n, float(n))
        lam = _table2(2.0 * np.pi * np.minimum(kk, n - kk) / n)       # cos is even about pi: theta reduced to [0, pi] in integers
    elif bc == NEUMANN:
        m = ((2 * i + 1) * k) % (4 * n)
        Phi = np.cos(np.pi * m.astype(np.float64) / (2 * n))
        w = np.full(n, n / 2.0)
        w[0] = float(n)
        lam = _table2(np.pi * kk / n)
    elif bc == DIRICHLET:
        m = ((2 * i + 1) * (k + 1)) % (4 * n)
        Phi = np.sin(np.pi * m.astype(np.float64) / (2 * n))
        w = np.full(n, n / 2.0)
        w[n - 1] = float(n)
        lam = _table2(np.pi * (kk + 1.0) / n)
    else:
        raise ValueError(f"unknown boundary condition {bc}")
    return Phi, w, lam


def forward_axis(g: np.ndarray, axis: int, bc: int) -> np.ndarray:
    """Unnormalised forward transform along ``axis``: ``ghat_k = sum_i g_i conj(phi_k(i))``.

    Exactly eq. 6 (periodic, DFT), eq. 7 (Neumann, DCT-II = "DCT10") or eq. 9 (Dirichlet,
    DST-II = "DST10") -- R2, R3: no normalisation in the forward direction.
    """
    Phi, _, _ = basis(g.shape[axis], bc)
    M = np.conj(Phi)  # M[i, k]
    if np.iscomplexobj(M) and not np.iscomplexobj(g):
        g = g.astype(np.complex128)
    out = np.moveaxis(np.moveaxis(g, axis, -1) @ M, -1, axis)
    return np.ascontiguousarray(out)


def inverse_axis(ghat: np.ndarray, axis: int, bc: int) -> np.ndarray:
    """Inverse of :func:`forward_axis`: ``g_i = sum_k ghat_k phi_k(i) / w_k``.

    For Neumann this is eq. 8 (DCT-III = "DCT01", the 1/2 on the k=0 term is w_0 = 2 w_k),
    for Dirichlet the corrected eq. 10 (DST-III = "DST01", R6: sin not cos, the 1/2 on the
    last term), both times 2/n; for periodic the inverse DFT with 1/n.
    """
    Phi, w, _ = basis(ghat.shape[axis], bc)
    M = (Phi / w[None, :]).T  # M[k, i]
    if np.iscomplexobj(M) and not np.iscomplexobj(ghat):
        ghat = ghat.astype(np.complex128)
    out = np.moveaxis(np.moveaxis(ghat, axis, -1) @ M, -1, axis)
    return np.ascontiguousarray(out)


# --------------------------------------------------------------------------------------
# tridiagonal solves (axis 0 of the arrays is the unknown index; the rest is a batch)
# --------------------------------------------------------------------------------------
def thomas(a, b, c, r):
    """Textbook Thomas algorithm, PAPER.md:224-248 (Algorithm 1; R9 for the garbled lines).

    ``a[k]`` sub-, ``b[k]`` main, ``c[k]`` super-diagonal of row k (``a[0]``, ``c[n-1]`` unused),
    ``r`` right-hand side, all with the unknown index on axis 0; any trailing batch shape.
    No pivoting.

        beta = b_0 ; x_0 = r_0 / beta
        for k = 1..n-1:  gamma_k = c_{k-1} / beta
                         beta    = b_k - a_k gamma_k
                         x_k     = (r_k - a_k x_{k-1}) / beta
        for k = n-2..0:  x_k = x_k - gamma_{k+1} x_{k+1}
    """
    n = r.shape[0]
    x = np.empty_like(r)
    gamma = np.empty_like(b)
    beta = b[0].copy()
    x[0] = r[0] / beta
    for k in range(1, n):
        gamma[k] = c[k - 1] / beta
        beta = b[k] - a[k] * gamma[k]
        x[k] = (r[k] - a[k] * x[k - 1]) / beta
    for k in range(n - 2, -1, -1):
        x[k] = x[k] - gamma[k + 1] * x[k + 1]
    return x


def z_coefficients(nz: int, bc_z: int, s, dtype=np.float64):
    """Three-value Toeplitz coefficients of Algorithm 2 (R10) expanded to
    full diagonals: ``T = L_z + s I``.  Interior diagonal ``-2 + s``, off-diagonals 1,
    first / last diagonal ``-1 + s`` (Neumann), ``-3 + s`` (Dirichlet), ``-2 + s`` (periodic;
    the cyclic corners are handled by the caller).
    """
    s = np.asarray(s, dtype=dtype)
    shape = (nz,) + s.shape
    b = np.empty(shape, dtype=dtype)
    b[:] = -2.0 + s
    if bc_z == NEUMANN:
        b[0] = -1.0 + s
        b[nz - 1] = -1.0 + s
    elif bc_z == DIRICHLET:
        b[0] = -3.0 + s
        b[nz - 1] = -3.0 + s
    a = np.ones(shape, dtype=dtype)
    c = np.ones(shape, dtype=dtype)
    return a, b, c


def cyclic_sherman_morrison(a, b, c, r):
    """Cyclic tridiagonal solve by the Sherman-Morrison formula -- "break down the periodic
    boundary condition to two solves" (R12).

    The cyclic matrix is ``T`` = tridiag(a, b, c) plus the corners ``T[0, n-1] = a_0`` and
    ``T[n-1, 0] = c_{n-1}``.  Write ``T = T' + w v^T`` with
        w = (gamma, 0, .., 0, c_{n-1})^T,  v = (1, 0, .., 0, a_0 / gamma)^T,  gamma = -b_0,
        T' = T without corners, b'_0 = b_0 - gamma, b'_{n-1} = b_{n-1} - c_{n-1} a_0 / gamma.
    Then  x = T'^-1 r,  q = T'^-1 w,  u = x - q (v.x) / (1 + v.q).
    """
    n = r.shape[0]
    gamma = -b[0]
    bp = b.copy()
    bp[0] = b[0] - gamma
    bp[n - 1] = b[n - 1] - c[n - 1] * a[0] / gamma
    w = np.zeros_like(b)
    w[0] = gamma
    w[n - 1] = c[n - 1]
    x = thomas(a, bp, c, r)
    q = thomas(a, bp, c, w)
    vx = x[0] + (a[0] / gamma) * x[n - 1]
    vq = q[0] + (a[0] / gamma) * q[n - 1]
    return x - q * (vx / (1.0 + vq))


def solve_zero_mode(r, bc_z: int):
    """The singular (kx, ky) = (0, 0) system, ``s = 0``, z periodic or Neumann (R11).

    ``T = L_z`` has the null vector 1.  (i) ``r <- r - mean(r)`` -- this is the paper's
    "integrate the source term over the volume and subtract it", since every other mode is
    mean-free; (ii) the paper's default, "keeping the corner value ... fixed": pin ``x_0 = 0``,
    drop row and column 0 and run Thomas on the remaining ``n-1`` rows; (iii) shift to zero
    mean, which selects the minimum-norm solution ``A^+ f`` and fixes the free constant.
    ``r`` is a 1-D array (length nz), real or complex.
    """
    n = r.shape[0]
    r = r - r.mean()
    x = np.zeros_like(r)
    if n > 1:
        m = n - 1
        real = np.real(r).dtype
        a = np.ones(m, dtype=real)
        c = np.ones(m, dtype=real)
        b = np.full(m, -2.0, dtype=real)
        if bc_z == NEUMANN:
            b[m - 1] = -1.0
        # periodic: dropping index 0 also drops both cyclic corners -> plain tridiagonal
        x[1:] = thomas(a, b, c, r[1:])
    return x - x.mean()


# --------------------------------------------------------------------------------------
# the whole solve
# --------------------------------------------------------------------------------------
def is_singular(bc) -> bool:
    """All three axes periodic or Neumann -> constants are in the null space."""
    return all(b in (PERIODIC, NEUMANN) for b in bc)


def solve(f: np.ndarray, h, bc, zdtype=np.float64) -> np.ndarray:
    """``u`` with ``A u = f`` (zero-mean ``u`` and mean-projected ``f`` if singular).

    f   : real array (nz, ny, nx)
    h   : (dx, dy, dz)
    bc  : (bc_x, bc_y, bc_z), each PERIODIC / NEUMANN / DIRICHLET (R14: one per axis)
    """
    f = np.asarray(f, dtype=np.float64)
    nz, ny, nx = f.shape
    dx, dy, dz = (float(v) for v in h)
    bx, by, bz = bc

    # 1. forward transforms, x then y (Table 1)
    fh = forward_axis(f, 2, bx)
    fh = forward_axis(fh, 1, by)

    # 2. one tridiagonal system in z per (kx, ky): T = L_z + s I,
    #    s = dz^2 (lam_x/dx^2 + lam_y/dy^2), rhs dz^2 fhat   (Table 2; R8)
    _, _, lamx = basis(nx, bx)
    _, _, lamy = basis(ny, by)
    s = dz * dz * (lamx[None, :] / (dx * dx) + lamy[:, None] / (dy * dy))  # (ny, nx)
    cdtype = np.result_type(zdtype, np.complex64) if np.iscomplexobj(fh) else zdtype
    rhs = (dz * dz) * fh.astype(cdtype)
    singular = is_singular(bc)
    s_work = s.astype(zdtype).copy()
    if singular:
        s_work[0, 0] = -1.0  # placeholder so the batched solve stays finite; overwritten below
    a, b, c = z_coefficients(nz, bz, s_work, dtype=zdtype)
    if bz == PERIODIC:
        uh = cyclic_sherman_morrison(a, b, c, rhs)
    else:
        uh = thomas(a, b, c, rhs)
    if singular:
        uh[:, 0, 0] = solve_zero_mode(rhs[:, 0, 0], bz)
    uh = uh.astype(np.complex128 if np.iscomplexobj(uh) else np.float64)

    # 3. inverse transforms, y then x
    u = inverse_axis(uh, 1, by)
    u = inverse_axis(u, 2, bx)
    if np.iscomplexobj(u):
        scale = max(float(np.max(np.abs(u.real))), np.finfo(np.float64).tiny)
        assert float(np.max(np.abs(u.imag))) <= 1e-12 * scale + 1e-300, "imaginary residue"
        u = u.real
    return np.ascontiguousarray(u)


# --------------------------------------------------------------------------------------
# the operator itself, for residual checks and brute force
# --------------------------------------------------------------------------------------
def fold_dirichlet(f: np.ndarray, h, bc, faces: dict) -> np.ndarray:
    """Non-homogeneous Dirichlet values moved to the right-hand side: with the ghost cell
    linearly extrapolated through the face value g, u_ghost = 2 g - u_0, the stencil of a boundary cell
    reads (u_1 - 3 u_0)/h^2 + 2 g/h^2 = f_0, i.e. the homogeneous operator with  f_0 <- f_0 - 2 g/h^2.

    ``faces`` maps (axis, side) -- axis in 'xyz', side 0 (lower face) or 1 (upper face) -- to the array of
    face values: shape (nz, ny) for x faces, (nz, nx) for y faces, (ny, nx) for z faces.  Returns a new
    array; ``f`` has shape (nz, ny, nx).  Every axis named must be Dirichlet."""
    out = np.array(f, dtype=np.float64, copy=True)
    nz, ny, nx = out.shape
    for (axis, side), g in faces.items():
        a = "xyz".index(axis)
        if bc[a] != DIRICHLET:
            raise ValueError(f"axis {axis} is not Dirichlet")
        c = 2.0 / (h[a] * h[a])
        g = np.asarray(g, dtype=np.float64)
        if axis == "x":
            assert g.shape == (nz, ny)
            out[:, :, nx - 1 if side else 0] -= c * g
        elif axis == "y":
            assert g.shape == (nz, nx)
            out[:, ny - 1 if side else 0, :] -= c * g
        else:
            assert g.shape == (ny, nx)
            out[nz - 1 if side else 0, :, :] -= c * g
    return out


def apply_A(u: np.ndarray, h, bc) -> np.ndarray:
    """``A u`` by the 7-point stencil of eq. 3 with the homogeneous boundary
    rows of :func:`lap1d`, written with shifted slices (no matrix)."""
    u = np.asarray(u, dtype=np.float64)
    out = np.zeros_like(u)
    for axis, (hh, b) in zip((2, 1, 0), zip(h, bc)):
        n = u.shape[axis]
        um = np.moveaxis(u, axis, 0)
        lo = np.empty_like(um)  # u_{i-1}
        hi = np.empty_like(um)  # u_{i+1}
        lo[1:] = um[:-1]
        hi[:-1] = um[1:]
        if b == PERIODIC:
            lo[0] = um[n - 1]
            hi[n - 1] = um[0]
        elif b == NEUMANN:
            lo[0] = um[0]
            hi[n - 1] = um[n - 1]
        elif b == DIRICHLET:
            lo[0] = -um[0]
            hi[n - 1] = -um[n - 1]
        else:
            raise ValueError(b)
        out += np.moveaxis((lo - 2.0 * um + hi) / (hh * hh), 0, axis)
    return out


def stencil_at(u_nbrs: np.ndarray, h) -> np.ndarray:
    """Eq. 3 at sampled points, one by one: ``u_nbrs[p] = (u_c, u_xm, u_xp, u_ym, u_yp, u_zm, u_zp)``
    with ghost values already substituted by the caller per :func:`lap1d`'s rules."""
    dx, dy, dz = h
    uc = u_nbrs[:, 0]
    return ((u_nbrs[:, 1] - 2 * uc + u_nbrs[:, 2]) / (dx * dx)
            + (u_nbrs[:, 3] - 2 * uc + u_nbrs[:, 4]) / (dy * dy)
            + (u_nbrs[:, 5] - 2 * uc + u_nbrs[:, 6]) / (dz * dz))


def dense_A(shape, h, bc) -> np.ndarray:
    """Kronecker-sum assembly of the full matrix (eq. 3-4), for brute force on tiny grids.
    Row / column index = i + nx (j + ny k)."""
    nz, ny, nx = shape
    dx, dy, dz = h
    Lx = lap1d(nx, bc[0]) / (dx * dx)
    Ly = lap1d(ny, bc[1]) / (dy * dy)
    Lz = lap1d(nz, bc[2]) / (dz * dz)
    Ix, Iy, Iz = np.eye(nx), np.eye(ny), np.eye(nz)
    return (np.kron(Iz, np.kron(Iy, Lx)) + np.kron(Iz, np.kron(Ly, Ix))
            + np.kron(Lz, np.kron(Iy, Ix)))
