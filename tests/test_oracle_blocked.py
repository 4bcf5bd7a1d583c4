"""The block-by-block driver of tests/oracle_blocked.py must give what ``po.solve`` gives on the whole array
(it is what the full-size GPU parity tests of configs 4 and 5 compare against)."""
import numpy as np
import pytest

from oracle import poisson_oracle as po
from oracle_blocked import oracle_solve_blocked, rel_err_blocked

N, D, P = po.NEUMANN, po.DIRICHLET, po.PERIODIC


@pytest.mark.parametrize("bc", [(D, D, D), (N, N, D), (N, D, N), (D, N, P)])
@pytest.mark.parametrize("blocks", [(16, 32), (3, 5), (1, 1)])
def test_blocked_driver_equals_whole_array_solve(bc, blocks):
    shape, h = (11, 13, 10), (0.2, 0.15, 0.4)
    f = np.random.default_rng(5).standard_normal(shape)
    ref = po.solve(f, h, bc)
    got = oracle_solve_blocked(f.copy(), h, bc, zblock=blocks[0], yblock=blocks[1])
    # same functions on sub-blocks: identical up to the BLAS's blocking of the matrix products
    assert rel_err_blocked(got, ref, zblock=4) <= 1e-14


def test_blocked_driver_refuses_what_it_does_not_cover():
    f = np.zeros((4, 4, 4))
    with pytest.raises(AssertionError):
        oracle_solve_blocked(f, (1, 1, 1), (P, N, D))
    with pytest.raises(AssertionError):
        oracle_solve_blocked(f, (1, 1, 1), (N, N, N))
