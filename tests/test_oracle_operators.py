"""Pins for the 1-D operators and eigenpairs of oracle/poisson_oracle.py.

What fixes them (not the oracle itself): Table 2 of the paper typed out
here, the stencil of eq. 3 applied by explicit Python loops, and the
orthogonality norms that the 1/2 terms of eq. 8 / eq. 10 encode."""
import math

import numpy as np
import pytest

from oracle import poisson_oracle as po

P, N, D = po.PERIODIC, po.NEUMANN, po.DIRICHLET


def table2(bc, k, n):
    """PAPER.md:200-206, typed literally."""
    if bc == P:
        return -2 + 2 * math.cos(2 * k * math.pi / n)
    if bc == N:
        return -2 + 2 * math.cos(k * math.pi / n)
    return -2 + 2 * math.cos((k + 1) * math.pi / n)


def stencil_loop(u, bc):
    """(L u)_i = u_{i-1} - 2 u_i + u_{i+1} with ghost cells per PAPER.md:126, 142, 163."""
    n = len(u)
    out = np.zeros(n, dtype=u.dtype)
    for i in range(n):
        if bc == P:
            lo, hi = u[(i - 1) % n], u[(i + 1) % n]
        else:
            ghost = (lambda v: v) if bc == N else (lambda v: -v)   # mirror / 2*0 - v
            lo = u[i - 1] if i > 0 else ghost(u[0])
            hi = u[i + 1] if i < n - 1 else ghost(u[n - 1])
        out[i] = lo - 2 * u[i] + hi
    return out


@pytest.mark.parametrize("bc", [P, N, D])
@pytest.mark.parametrize("n", [2, 3, 5, 6, 7, 8, 16, 33])
def test_lap1d_is_the_stencil(bc, n):
    rng = np.random.default_rng(n * 10 + bc)
    u = rng.standard_normal(n)
    np.testing.assert_allclose(po.lap1d(n, bc) @ u, stencil_loop(u, bc), rtol=0, atol=1e-14)


@pytest.mark.parametrize("bc", [P, N, D])
@pytest.mark.parametrize("n", [4, 5, 6, 7, 8, 16, 31, 64])
def test_table2_eigenpairs(bc, n):
    Phi, w, lam = po.basis(n, bc)
    lam_paper = np.array([table2(bc, k, n) for k in range(n)])
    np.testing.assert_allclose(lam, lam_paper, rtol=0, atol=4e-15)     # |lam| <= 4: a few eps of 4 (R27: -4 sin^2 against the printed -2 + 2 cos)
    for k in range(n):
        lhs = stencil_loop(Phi[:, k].copy(), bc)
        np.testing.assert_allclose(lhs, lam_paper[k] * Phi[:, k], rtol=0, atol=2e-13)


@pytest.mark.parametrize("bc", [P, N, D])
@pytest.mark.parametrize("n", [512, 2048, 16384])
def test_table2_long_axes_without_cancellation(bc, n):
    """Reading R27: the oracle evaluates Table 2's -2 + 2 cos(theta) as -4 sin^2(theta / 2).  Typed as printed but in
    80-bit arithmetic it must agree within that evaluation's own error: |lam - printed| <= 4 eps64 |printed| + 4 eps80
    (the 80-bit sum -2 + 2 cos carries an absolute rounding error of a few eps80 = 1.1e-19: 2e-13 relative on the lowest
    mode of n = 2048).  The printed form in fp64 misses that by three orders (ten digits at n = 2048): the error the
    identity removes."""
    if np.finfo(np.longdouble).eps > 2e-19:
        # no 80-bit long double on this host: the same pin in 60-digit decimal arithmetic (never skipped, so that
        # R27 cannot lose its pin silently)
        import hp_trig
        from decimal import Decimal
        _, _, lam = po.basis(n, bc) if n <= 2048 else (None, None, po._table2(
            {P: 2.0 * np.pi * np.minimum(np.arange(n, dtype=np.float64), n - np.arange(n, dtype=np.float64)) / n,
             N: np.pi * np.arange(n, dtype=np.float64) / n, D: np.pi * (np.arange(n, dtype=np.float64) + 1.0) / n}[bc]))
        for k in list(range(0, 64)) + list(range(64, n, 97)) + [n - 1]:
            printed = hp_trig.table2_printed(bc, k, n)
            assert abs(Decimal(float(lam[k])) - printed) <= 4 * Decimal(2.0 ** -52) * abs(printed) + Decimal(1e-30), k
        return
    if n <= 2048:
        _, _, lam = po.basis(n, bc)
    else:                                                  # (the basis matrix of 16384^2 entries is not needed here)
        kq = np.arange(n, dtype=np.float64)
        lam = po._table2({P: 2.0 * np.pi * np.minimum(kq, n - kq) / n, N: np.pi * kq / n, D: np.pi * (kq + 1.0) / n}[bc])
    k = np.arange(n, dtype=np.longdouble)
    pi = np.longdouble("3.14159265358979323846264338327950288")
    theta = {P: 2 * k * pi / n, N: k * pi / n, D: (k + 1) * pi / n}[bc]
    printed = -2 + 2 * np.cos(theta)                       # PAPER.md:200-206, in long double
    nz = np.abs(printed) > 0
    err = np.abs(lam[nz].astype(np.longdouble) - printed[nz])
    bound = 4 * np.finfo(np.float64).eps * np.abs(printed[nz]) + 4 * np.finfo(np.longdouble).eps
    assert np.all(err <= bound), float((err / bound).max())
    assert np.all(np.abs(lam[~nz]) <= 4 * np.finfo(np.longdouble).eps)
    rel = err / np.abs(printed[nz])
    # the printed form in fp64 loses digits on the low modes of a long axis
    kd = np.arange(n, dtype=np.float64)
    thd = {P: 2 * kd * np.pi / n, N: kd * np.pi / n, D: (kd + 1) * np.pi / n}[bc]
    printed64 = -2.0 + 2.0 * np.cos(thd)
    rel64 = np.abs((printed64[nz].astype(np.longdouble) - printed[nz]) / printed[nz])
    if n >= 2048:
        assert float(rel64.max()) > 1e-12 and float(rel64.max()) > 10 * float(rel.max())


@pytest.mark.parametrize("bc", [P, N, D])
@pytest.mark.parametrize("n", [4, 5, 8, 9, 32])
def test_basis_orthogonality_and_norms(bc, n):
    Phi, w, _ = po.basis(n, bc)
    G = Phi.conj().T @ Phi
    # squared norms typed out: n for periodic; n/2 except the constant (Neumann k=0) and the
    # alternating (Dirichlet k=n-1) vectors, which have n
    w_ref = np.full(n, float(n) if bc == P else n / 2)
    if bc == N:
        w_ref[0] = n
    if bc == D:
        w_ref[n - 1] = n
    np.testing.assert_allclose(G, np.diag(w_ref), rtol=0, atol=1e-12)
    np.testing.assert_allclose(w, w_ref)


def test_basis_entries_literal():
    """phi_k(i) against direct evaluation of the formulas in eq. 6, 7, 9."""
    n = 7
    for bc, fn in ((P, lambda i, k: complex(math.cos(2 * math.pi * k * i / n), math.sin(2 * math.pi * k * i / n))),
                   (N, lambda i, k: math.cos((i + 0.5) * k * math.pi / n)),
                   (D, lambda i, k: math.sin((i + 0.5) * (k + 1) * math.pi / n))):
        Phi, _, _ = po.basis(n, bc)
        for i in range(n):
            for k in range(n):
                assert abs(Phi[i, k] - fn(i, k)) < 1e-14


@pytest.mark.parametrize("bc", [(P, N, D), (D, P, N), (N, D, P), (P, P, P), (N, N, N), (D, D, D)])
def test_apply_A_matches_dense(bc):
    shape, h = (5, 4, 6), (0.3, 0.2, 0.45)
    rng = np.random.default_rng(1)
    u = rng.standard_normal(shape)
    A = po.dense_A(shape, h, bc)
    np.testing.assert_allclose(po.apply_A(u, h, bc).ravel(), A @ u.ravel(), rtol=0, atol=1e-11)


def test_dense_A_row_is_eq3():
    """One interior row of the assembled matrix against eq. 3 typed out."""
    shape, h = (4, 5, 6), (0.5, 0.25, 0.125)
    nz, ny, nx = shape
    A = po.dense_A(shape, h, (P, N, D))
    i, j, k = 2, 3, 1
    row = A[i + nx * (j + ny * k)]
    expect = {}
    expect[(i, j, k)] = -2 / h[0] ** 2 - 2 / h[1] ** 2 - 2 / h[2] ** 2
    expect[(i - 1, j, k)] = expect[(i + 1, j, k)] = 1 / h[0] ** 2
    expect[(i, j - 1, k)] = expect[(i, j + 1, k)] = 1 / h[1] ** 2
    expect[(i, j, k - 1)] = expect[(i, j, k + 1)] = 1 / h[2] ** 2
    ref = np.zeros_like(row)
    for (ii, jj, kk), v in expect.items():
        ref[ii + nx * (jj + ny * kk)] = v
    np.testing.assert_allclose(row, ref, rtol=0, atol=1e-12)
