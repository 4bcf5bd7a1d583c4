"""Pins for the tridiagonal pieces: dense ``numpy.linalg.solve`` / ``pinv`` on the assembled
matrices (PAPER.md:224-284 Algorithms 1-2; PAPER.md:216 Sherman-Morrison)."""
import numpy as np
import pytest

from oracle import poisson_oracle as po

P, N, D = po.PERIODIC, po.NEUMANN, po.DIRICHLET


def assemble(a, b, c, cyclic=False):
    n = len(b)
    T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    if cyclic:
        T[0, n - 1] += a[0]
        T[n - 1, 0] += c[n - 1]
    return T


@pytest.mark.parametrize("n", [1, 2, 3, 8, 33, 64])
def test_thomas_general_vs_dense(n):
    rng = np.random.default_rng(n)
    a, c = rng.uniform(0.5, 1.5, n), rng.uniform(0.5, 1.5, n)
    b = -(np.abs(a) + np.abs(c) + rng.uniform(0.1, 2.0, n))
    r = rng.standard_normal(n)
    x = po.thomas(a, b, c, r)
    np.testing.assert_allclose(x, np.linalg.solve(assemble(a, b, c), r), rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("bc_z", [N, D])
@pytest.mark.parametrize("n", [2, 3, 7, 32, 64])
def test_toeplitz_coefficients_and_batched_thomas(bc_z, n):
    rng = np.random.default_rng(10 * n + bc_z)
    s = -rng.uniform(1e-3, 8.0, size=(3, 4))
    a, b, c = po.z_coefficients(n, bc_z, s)
    r = rng.standard_normal((n, 3, 4)) + 1j * rng.standard_normal((n, 3, 4))
    x = po.thomas(a, b, c, r)
    Lz = po.lap1d(n, bc_z)
    for j in range(3):
        for i in range(4):
            T = Lz + s[j, i] * np.eye(n)
            np.testing.assert_allclose(assemble(a[:, j, i], b[:, j, i], c[:, j, i]), T, rtol=0, atol=1e-14)
            np.testing.assert_allclose(x[:, j, i], np.linalg.solve(T, r[:, j, i]), rtol=1e-11, atol=1e-12)


@pytest.mark.parametrize("n", [3, 4, 9, 32, 64])
def test_cyclic_sherman_morrison_vs_dense(n):
    rng = np.random.default_rng(n + 77)
    s = -rng.uniform(1e-3, 8.0, size=(5,))
    a, b, c = po.z_coefficients(n, P, s)
    r = rng.standard_normal((n, 5)) + 1j * rng.standard_normal((n, 5))
    x = po.cyclic_sherman_morrison(a, b, c, r)
    Lz = po.lap1d(n, P)
    for i in range(5):
        T = Lz + s[i] * np.eye(n)
        np.testing.assert_allclose(assemble(a[:, i], b[:, i], c[:, i], cyclic=True), T, rtol=0, atol=1e-14)
        np.testing.assert_allclose(x[:, i], np.linalg.solve(T, r[:, i]), rtol=1e-11, atol=1e-12)


def test_cyclic_general_coefficients_vs_dense():
    n = 12
    rng = np.random.default_rng(5)
    a, c = rng.uniform(0.5, 1.5, n), rng.uniform(0.5, 1.5, n)
    b = -(a + c + rng.uniform(0.5, 2.0, n))
    r = rng.standard_normal(n)
    x = po.cyclic_sherman_morrison(a, b, c, r)
    np.testing.assert_allclose(x, np.linalg.solve(assemble(a, b, c, cyclic=True), r), rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("bc_z", [P, N])
@pytest.mark.parametrize("n", [2, 3, 8, 33, 128])
def test_zero_mode_is_the_pseudo_inverse(bc_z, n):
    rng = np.random.default_rng(n + 5)
    r = rng.standard_normal(n) + 1j * rng.standard_normal(n) + 3.0      # deliberately not mean-free
    x = po.solve_zero_mode(r, bc_z)
    Lz = po.lap1d(n, bc_z)
    np.testing.assert_allclose(x, np.linalg.pinv(Lz) @ r, rtol=0, atol=1e-10 * n)
    assert abs(x.mean()) < 1e-13 * n
    np.testing.assert_allclose(Lz @ x, r - r.mean(), rtol=0, atol=1e-11 * n)
    # a constant added to r changes nothing
    np.testing.assert_allclose(po.solve_zero_mode(r + 11.0, bc_z), x, rtol=0, atol=1e-11 * n)


def test_thomas_longdouble_runs_and_is_closer():
    n = 256
    s = np.array([-5.9e-7])
    rng = np.random.default_rng(1)
    r = rng.standard_normal((n, 1))
    a, b, c = po.z_coefficients(n, N, s, dtype=np.longdouble)
    x_ld = po.thomas(a, b, c, r.astype(np.longdouble))
    a, b, c = po.z_coefficients(n, N, s)
    x_d = po.thomas(a, b, c, r)
    rel = np.max(np.abs(x_d - x_ld.astype(np.float64))) / np.max(np.abs(x_d))
    assert rel < 1e-8          # fp64 Thomas is only ~1e-10 accurate here (DESIGN.md precision hazards)
