"""The oracle's solve applied block by block, for grids whose whole-array temporaries do not fit the host
(BASELINE.json configs 4 and 5: 2^30 and 2^29 points).

This blocks the TEST, not the oracle: every arithmetic step is a call of ``oracle.poisson_oracle``'s own
functions (`forward_axis`, `basis`, `z_coefficients`, `thomas` / `cyclic_sherman_morrison`, `inverse_axis`)
in the order and with the formulas of ``po.solve`` -- x and y transforms are independent per z plane, the z
systems independent per (kx, ky), so slabs of planes and slabs of modes give bit-identical results
(tests/test_oracle_blocked.py checks that on the CPU).  Non-singular problems only."""
import numpy as np

from oracle import poisson_oracle as po


def oracle_solve_blocked(f, h, bc, zblock=16, yblock=32, zdtype=np.float64):
    """In place: on return ``f`` holds u.  ``f``: float64 (nz, ny, nx), real transforms on x and y (no periodic
    x / y axis: the spectrum stays real and the array can be reused)."""
    nz, ny, nx = f.shape
    dx, dy, dz = (float(v) for v in h)
    bx, by, bz = bc
    assert bx != po.PERIODIC and by != po.PERIODIC, "blocked driver: real transforms only"
    assert not po.is_singular(bc)
    # 1. forward transforms x then y, plane slab by plane slab (po.solve step 1)
    for k0 in range(0, nz, zblock):
        sl = slice(k0, min(k0 + zblock, nz))
        f[sl] = po.forward_axis(po.forward_axis(f[sl], 2, bx), 1, by)
    # 2. one tridiagonal system per (kx, ky), mode slab by mode slab (po.solve step 2)
    _, _, lamx = po.basis(nx, bx)
    _, _, lamy = po.basis(ny, by)
    for j0 in range(0, ny, yblock):
        js = slice(j0, min(j0 + yblock, ny))
        s = dz * dz * (lamx[None, :] / (dx * dx) + lamy[js, None] / (dy * dy))
        a, b, c = po.z_coefficients(nz, bz, s.astype(zdtype), dtype=zdtype)
        rhs = (dz * dz) * f[:, js, :].astype(zdtype)
        uh = po.cyclic_sherman_morrison(a, b, c, rhs) if bz == po.PERIODIC else po.thomas(a, b, c, rhs)
        f[:, js, :] = uh.astype(np.float64)
    # 3. inverse transforms y then x (po.solve step 3)
    for k0 in range(0, nz, zblock):
        sl = slice(k0, min(k0 + zblock, nz))
        f[sl] = po.inverse_axis(po.inverse_axis(f[sl], 1, by), 2, bx)
    return f


def rel_err_blocked(u, ref, zblock=16):
    """max|u - ref| / max|ref| without whole-array temporaries."""
    num = den = 0.0
    for k0 in range(0, ref.shape[0], zblock):
        sl = slice(k0, k0 + zblock)
        num = max(num, float(np.max(np.abs(u[sl] - ref[sl]))))
        den = max(den, float(np.max(np.abs(ref[sl]))))
    return num / max(den, np.finfo(np.float64).tiny)
