"""Pins for the whole oracle solve: dense brute force for all 27 boundary-condition
combinations, closed-form single-mode solutions, the 7-point residual, the singular-case
invariants, and structural symmetries."""
import itertools
import math

import numpy as np
import pytest

from oracle import poisson_oracle as po

P, N, D = po.PERIODIC, po.NEUMANN, po.DIRICHLET
ALL27 = list(itertools.product((P, N, D), repeat=3))


def name(bc):
    return "".join(po.BC_NAMES[b] for b in bc)


@pytest.mark.parametrize("bc", ALL27, ids=name)
def test_brute_force_dense_all_27(bc):
    """A assembled by Kronecker sums (eq. 3-4) and solved by LAPACK, on a non-cubic,
    non-power-of-two, anisotropic grid (nx=6, ny=5, nz=7)."""
    shape, h = (7, 5, 6), (0.3, 0.2, 0.45)
    rng = np.random.default_rng(sum(b * 3 ** i for i, b in enumerate(bc)))
    f = rng.standard_normal(shape)
    A = po.dense_A(shape, h, bc)
    u = po.solve(f, h, bc)
    if po.is_singular(bc):
        ref = np.linalg.pinv(A) @ f.ravel()
    else:
        ref = np.linalg.solve(A, f.ravel())
    np.testing.assert_allclose(u.ravel(), ref, rtol=0, atol=2e-13 * np.max(np.abs(ref)) + 1e-15)


@pytest.mark.parametrize("bc", [(P, P, N), (N, D, P), (D, D, D), (P, N, D)], ids=name)
def test_brute_force_second_shape(bc):
    shape, h = (4, 12, 8), (1.0 / 8, 1.0 / 12, 0.5)
    rng = np.random.default_rng(42)
    f = rng.standard_normal(shape)
    A = po.dense_A(shape, h, bc)
    u = po.solve(f, h, bc)
    ref = (np.linalg.pinv(A) if po.is_singular(bc) else np.linalg.inv(A)) @ f.ravel()
    np.testing.assert_allclose(u.ravel(), ref, rtol=0, atol=2e-13 * np.max(np.abs(ref)))


def mode_1d(bc, n, k):
    i = np.arange(n)
    if bc == P:
        return np.cos(2 * math.pi * k * i / n), -2 + 2 * math.cos(2 * k * math.pi / n)
    if bc == N:
        return np.cos((i + 0.5) * k * math.pi / n), -2 + 2 * math.cos(k * math.pi / n)
    return np.sin((i + 0.5) * (k + 1) * math.pi / n), -2 + 2 * math.cos((k + 1) * math.pi / n)


@pytest.mark.parametrize("bc", ALL27, ids=name)
def test_closed_form_single_modes(bc):
    """f = phi_kx (x) phi_ky (x) phi_kz  =>  u = f / (lx/dx^2 + ly/dy^2 + lz/dz^2)  exactly
    (Table 2), including k = 0, Nyquist and k = n-1."""
    nx, ny, nz = 16, 8, 12
    h = (1.0 / 16, 0.1, 0.07)
    for kx, ky, kz in [(0, 0, 1), (1, 0, 0), (nx // 2, ny // 2, nz // 2), (nx - 1, ny - 1, nz - 1), (3, 2, 5)]:
        gx, lx = mode_1d(bc[0], nx, kx)
        gy, ly = mode_1d(bc[1], ny, ky)
        gz, lz = mode_1d(bc[2], nz, kz)
        lam = lx / h[0] ** 2 + ly / h[1] ** 2 + lz / h[2] ** 2
        f = gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
        if abs(lam) < 1e-9:
            continue
        u = po.solve(f, h, bc)
        np.testing.assert_allclose(u, f / lam, rtol=0, atol=1e-13 * np.max(np.abs(f / lam)))


@pytest.mark.parametrize("bc", ALL27, ids=name)
def test_residual_and_singular_invariants(bc):
    shape, h = (10, 12, 16), (1.0 / 16, 1.0 / 12, 0.13)
    rng = np.random.default_rng(9)
    f = rng.standard_normal(shape)
    u = po.solve(f, h, bc)
    target = f - f.mean() if po.is_singular(bc) else f
    res = po.apply_A(u, h, bc) - target
    assert np.max(np.abs(res)) <= 1e-10 * np.max(np.abs(f))
    if po.is_singular(bc):
        assert abs(u.mean()) <= 1e-14 * np.max(np.abs(u))
        u2 = po.solve(f + 123.0, h, bc)                    # constants in f are projected out
        np.testing.assert_allclose(u2, u, rtol=0, atol=1e-11 * np.max(np.abs(u)))


def test_linearity_and_symmetries():
    shape, h, bc = (6, 8, 10), (0.1, 0.2, 0.3), (P, N, D)
    rng = np.random.default_rng(11)
    f1, f2 = rng.standard_normal(shape), rng.standard_normal(shape)
    u1, u2 = po.solve(f1, h, bc), po.solve(f2, h, bc)
    scale = np.max(np.abs(u1)) + np.max(np.abs(u2))
    np.testing.assert_allclose(po.solve(2 * f1 - 3 * f2, h, bc), 2 * u1 - 3 * u2, rtol=0, atol=1e-12 * scale)
    # translation along the periodic axis (x)
    np.testing.assert_allclose(po.solve(np.roll(f1, 3, axis=2), h, bc), np.roll(u1, 3, axis=2), rtol=0, atol=1e-12 * scale)
    # mirror along the Neumann (y) and Dirichlet (z) axes
    np.testing.assert_allclose(po.solve(f1[:, ::-1, :], h, bc), u1[:, ::-1, :], rtol=0, atol=1e-12 * scale)
    np.testing.assert_allclose(po.solve(f1[::-1, :, :], h, bc), u1[::-1, :, :], rtol=0, atol=1e-12 * scale)
    # swapping x and y (with BCs and spacings) transposes the result
    fT = np.ascontiguousarray(np.swapaxes(f1, 1, 2))
    uT = po.solve(fT, (h[1], h[0], h[2]), (bc[1], bc[0], bc[2]))
    np.testing.assert_allclose(uT, np.swapaxes(u1, 1, 2), rtol=0, atol=1e-12 * scale)


def test_z_axis_is_solved_like_the_others():
    """Rotating the axes (x->y->z->x) must give the rotated solution although z is solved by
    Thomas and x, y by transforms."""
    shape, h, bc = (8, 6, 10), (0.1, 0.2, 0.3), (N, D, P)
    f = np.random.default_rng(12).standard_normal(shape)
    u = po.solve(f, h, bc)
    fr = np.ascontiguousarray(np.transpose(f, (1, 2, 0)))            # new (z,y,x) = old (y,x,z)
    ur = po.solve(fr, (h[2], h[0], h[1]), (bc[2], bc[0], bc[1]))
    np.testing.assert_allclose(ur, np.transpose(u, (1, 2, 0)), rtol=0, atol=1e-12 * np.max(np.abs(u)))


def test_longdouble_z_option():
    shape, h, bc = (16, 8, 8), (0.1, 0.1, 0.05), (P, P, N)
    f = np.random.default_rng(13).standard_normal(shape)
    u = po.solve(f, h, bc)
    u_ld = po.solve(f, h, bc, zdtype=np.longdouble)
    assert u_ld.dtype == np.float64
    np.testing.assert_allclose(u_ld, u, rtol=0, atol=1e-12 * np.max(np.abs(u)))


@pytest.mark.parametrize("long_axis", ["x", "y"])
@pytest.mark.parametrize("bc_long", [P, N, D], ids=lambda b: "PND"[b])
def test_closed_form_low_modes_on_a_long_axis(long_axis, bc_long, monkeypatch):
    """Solve-level pin of reading R27: on a 2048-point transform axis the lowest modes have
    lam = -2 + 2 cos(theta) ~ -1e-5, and u = f / lam divides by it.  Expected values: Table 2 AS PRINTED,
    evaluated in 60-digit decimal arithmetic (tests/hp_trig.py -- neither the oracle's formula nor the host's long double).
    The oracle must be within 1e-13; with `_table2` put back to the printed form in fp64 it is not within 1e-11 (periodic axis: 2e-12) -- the
    cancellation R27 removes is visible at the level of the solve, and this test would catch its return.
    The z recurrence runs in long double (`zdtype`): with a shift this small the fp64 Thomas elimination itself loses
    eps / |s| ~ 1e-11 (precision hazards), which would hide what is being pinned; the shift it is given is
    still the fp64 value of `_table2`.  On a host without 80-bit long double the bounds are the fp64 recurrence's."""
    import hp_trig
    n = 2048
    h = (0.37, 0.37, 0.37)
    shape = (2, 2, n) if long_axis == "x" else (2, n, 2)
    bc = (bc_long, N, N) if long_axis == "x" else (N, bc_long, N)          # Neumann mode 0 (constant) on the short axes: lam = 0
    ks = [1, 2, 3] if bc_long != D else [0, 1, 2]                          # the three lowest non-zero eigenvalues
    i = np.arange(n)
    printed_form = lambda theta: -2.0 + 2.0 * np.cos(theta)                # noqa: E731  (the fp64 form R27 replaced)
    worst_new, worst_old = 0.0, 0.0
    for k in ks:
        g = mode_1d(bc_long, n, k)[0]
        f = np.broadcast_to(g[None, None, :] if long_axis == "x" else g[None, :, None], shape).copy()
        lam = float(hp_trig.table2_printed(bc_long, k, n)) / h[0] ** 2
        want = f / lam
        u = po.solve(f, h, bc, zdtype=np.longdouble)
        worst_new = max(worst_new, float(np.max(np.abs(u - want)) / np.max(np.abs(want))))
        with monkeypatch.context() as m:
            m.setattr(po, "_table2", printed_form)
            u_old = po.solve(f, h, bc, zdtype=np.longdouble)
        worst_old = max(worst_old, float(np.max(np.abs(u_old - want)) / np.max(np.abs(want))))
    if np.finfo(np.longdouble).eps < 2e-19:
        assert worst_new <= 1e-13, worst_new
        # (periodic theta = 2 pi k / n is twice the others: the printed form loses four times less there)
        assert worst_old > (2e-12 if bc_long == P else 1e-11) and worst_old > 20 * worst_new, (worst_old, worst_new)
    else:
        assert worst_new <= 3e-11, worst_new
        assert worst_old > 3 * worst_new, (worst_old, worst_new)
