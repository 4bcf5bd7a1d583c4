"""Pins for ``oracle.poisson_oracle.stencil_at`` and for the neighbour gathering of
tests/stencil_sampling.py -- the checker behind the sampled-residual tests at BASELINE.json's two largest
configurations (tests/test_gpu_fullsize.py).

What fixes them (not themselves): eq. 3 typed out with explicit loops and ghost cells
(PAPER.md:126, 142, 163), ``dense_A`` (pinned by a typed row in test_oracle_solve.py) and ``apply_A``
(pinned against dense_A).  Three different spacings and a non-cubic grid: a swapped column, a swapped
spacing, a wrong ghost sign or a wrong wrap on any axis fails."""
import itertools

import numpy as np
import pytest

from oracle import poisson_oracle as po
import stencil_sampling as ss

P, N, D = po.PERIODIC, po.NEUMANN, po.DIRICHLET
H = (0.3, 0.07, 1.9)              # three different spacings (dx, dy, dz)
SHAPE = (5, 6, 7)                 # (nz, ny, nx), all different


def eq3_by_loops(u, h, bc, cells):
    """Eq. 3 at the given cells, ghost values substituted one at a time."""
    nz, ny, nx = u.shape
    dx, dy, dz = h

    def at(k, j, i):
        sign = 1.0
        for axis, (n, b) in enumerate(zip((nx, ny, nz), bc)):
            t = (i, j, k)[axis]
            if t < 0 or t >= n:
                if b == P:
                    t = t % n
                else:
                    t = 0 if t < 0 else n - 1
                    if b == D:
                        sign = -sign
                if axis == 0:
                    i = t
                elif axis == 1:
                    j = t
                else:
                    k = t
        return sign * u[k, j, i]

    out = []
    for k, j, i in cells:
        c = at(k, j, i)
        out.append((at(k, j, i - 1) - 2 * c + at(k, j, i + 1)) / dx ** 2
                   + (at(k, j - 1, i) - 2 * c + at(k, j + 1, i)) / dy ** 2
                   + (at(k - 1, j, i) - 2 * c + at(k + 1, j, i)) / dz ** 2)
    return np.array(out)


def all_cells(shape):
    k, j, i = np.meshgrid(*(np.arange(n) for n in shape), indexing="ij")
    return k.ravel(), j.ravel(), i.ravel()


@pytest.mark.parametrize("bc", list(itertools.product((P, N, D), repeat=3)))
def test_stencil_at_every_cell_matches_loops_and_apply_A(bc):
    rng = np.random.default_rng(sum(b * 3 ** a for a, b in enumerate(bc)))
    u = rng.standard_normal(SHAPE)
    idx = all_cells(SHAPE)
    nb = ss.gather_numpy(u, ss.neighbour_table(idx, SHAPE, bc))
    got = po.stencil_at(nb, H)
    want = eq3_by_loops(u, H, bc, list(zip(*idx)))
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)
    np.testing.assert_allclose(got, po.apply_A(u, H, bc)[idx], rtol=0, atol=1e-12)
    np.testing.assert_allclose(got, po.dense_A(SHAPE, H, bc) @ u.ravel(), rtol=0, atol=1e-12)


def test_stencil_at_columns_are_not_interchangeable():
    """u = x^2 / 2 has second difference 1 along x and 0 along y, z: only the (x-1, x+1) columns paired with dx
    give 1/dx^2 * dx^2 = 1 -- a column or spacing swap gives something else."""
    nz, ny, nx = 4, 5, 9
    x = (np.arange(nx) + 0.5) * H[0]
    u = np.broadcast_to(0.5 * x * x, (nz, ny, nx)).copy()
    idx = (np.array([1, 2]), np.array([2, 3]), np.array([3, 5]))          # interior cells
    nb = ss.gather_numpy(u, ss.neighbour_table(idx, u.shape, (N, N, N)))
    np.testing.assert_allclose(po.stencil_at(nb, H), [1.0, 1.0], rtol=0, atol=1e-12)
    for perm in ([0, 3, 4, 1, 2, 5, 6], [0, 5, 6, 3, 4, 1, 2]):           # x <-> y, x <-> z columns
        assert np.all(np.abs(po.stencil_at(nb[:, perm], H) - 1.0) > 0.1)


def test_sampled_cells_cover_faces_edges_and_corners():
    shape = (8, 9, 10)
    k, j, i = ss.sample_indices(shape, 3000, seed=1)
    on = [(k == 0) | (k == shape[0] - 1), (j == 0) | (j == shape[1] - 1), (i == 0) | (i == shape[2] - 1)]
    for a in on:
        assert a.sum() >= 900
    assert (on[0] & on[1]).any() and (on[1] & on[2]).any() and (on[0] & on[1] & on[2]).any()
    assert (~(on[0] | on[1] | on[2])).any()


@pytest.mark.parametrize("bc", [(P, P, N), (N, N, D), (D, D, D), (N, D, P)])
def test_sampled_residual_of_the_oracle_solution_is_at_rounding_level(bc):
    """The whole checker on the CPU: solve, gather sampled neighbours, residual -- and a corrupted solution fails."""
    shape, h = (12, 10, 14), (0.11, 0.13, 0.17)
    rng = np.random.default_rng(3)
    f = rng.standard_normal(shape)
    if po.is_singular(bc):
        f -= f.mean()
    u = po.solve(f, h, bc)
    idx = ss.sample_indices(shape, 600, seed=2)
    nb = ss.gather_numpy(u, ss.neighbour_table(idx, shape, bc))
    res = np.max(np.abs(po.stencil_at(nb, h) - f[idx]))
    assert res <= 1e-11 * np.max(np.abs(f))
    u[idx[0][0], idx[1][0], idx[2][0]] += 1e-6
    nb = ss.gather_numpy(u, ss.neighbour_table(idx, shape, bc))
    assert np.max(np.abs(po.stencil_at(nb, h) - f[idx])) > 1e-6
