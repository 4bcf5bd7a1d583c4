"""Pins for the transforms: eq. 6-10 evaluated literally with Python loops, the two worked
5-element examples the paper prints, and round trips."""
import math
import os

import numpy as np
import pytest

from oracle import makhoul as mk
from oracle import poisson_oracle as po

P, N, D = po.PERIODIC, po.NEUMANN, po.DIRICHLET
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def eq6(u):
    n = len(u)
    return np.array([sum(u[m] * complex(math.cos(2 * math.pi * k * m / n), -math.sin(2 * math.pi * k * m / n))
                         for m in range(n)) for k in range(n)])


def eq7(u):   # PAPER.md:128  DCT-II ("DCT10")
    n = len(u)
    return np.array([sum(u[m] * math.cos((m + 0.5) * k * math.pi / n) for m in range(n)) for k in range(n)])


def eq8(Y):   # PAPER.md:152  DCT-III ("DCT01")
    n = len(Y)
    return np.array([0.5 * Y[0] + sum(Y[m] * math.cos((k + 0.5) * m * math.pi / n) for m in range(1, n))
                     for k in range(n)])


def eq9(u):   # PAPER.md:165  DST-II ("DST10")
    n = len(u)
    return np.array([sum(u[m] * math.sin((m + 0.5) * (k + 1) * math.pi / n) for m in range(n)) for k in range(n)])


def eq10(Y, trig=math.sin):   # PAPER.md:176 as corrected by R6 (sin); trig=math.cos is "as printed"
    n = len(Y)
    return np.array([((-1) ** k) / 2 * Y[n - 1] + sum(Y[m] * trig((m + 1) * (k + 0.5) * math.pi / n)
                                                      for m in range(n - 1)) for k in range(n)])


@pytest.mark.parametrize("n", [2, 3, 4, 5, 8, 12, 17])
def test_forward_is_the_printed_definition(n):
    rng = np.random.default_rng(n)
    u = rng.standard_normal(n)
    np.testing.assert_allclose(po.forward_axis(u, 0, P), eq6(u), rtol=0, atol=1e-13)
    np.testing.assert_allclose(po.forward_axis(u, 0, N), eq7(u), rtol=0, atol=1e-13)
    np.testing.assert_allclose(po.forward_axis(u, 0, D), eq9(u), rtol=0, atol=1e-13)


@pytest.mark.parametrize("n", [2, 3, 4, 5, 8, 12, 17])
def test_inverse_is_eq8_eq10_times_2_over_n(n):
    rng = np.random.default_rng(100 + n)
    Y = rng.standard_normal(n)
    np.testing.assert_allclose(po.inverse_axis(Y, 0, N), (2.0 / n) * eq8(Y), rtol=0, atol=1e-13)
    np.testing.assert_allclose(po.inverse_axis(Y, 0, D), (2.0 / n) * eq10(Y), rtol=0, atol=1e-13)
    u = rng.standard_normal(n)
    np.testing.assert_allclose((2.0 / n) * eq8(eq7(u)), u, rtol=0, atol=1e-13)
    np.testing.assert_allclose((2.0 / n) * eq10(eq9(u)), u, rtol=0, atol=1e-13)


def test_eq10_with_cos_as_printed_is_not_an_inverse():
    """Documents reading R6: PAPER.md:176 prints cos; only sin inverts eq. 9."""
    u = np.random.default_rng(3).standard_normal(8)
    bad = (2.0 / 8) * eq10(eq9(u), trig=math.cos)
    assert np.max(np.abs(bad - u)) > 0.1


@pytest.mark.parametrize("bc", [P, N, D])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_round_trip_any_axis(bc, axis):
    rng = np.random.default_rng(7)
    g = rng.standard_normal((5, 6, 7))
    back = po.inverse_axis(po.forward_axis(g, axis, bc), axis, bc)
    np.testing.assert_allclose(np.real(back), g, rtol=0, atol=1e-13)
    assert np.max(np.abs(np.imag(back))) < 1e-13


def test_axis_transform_is_linewise():
    rng = np.random.default_rng(8)
    g = rng.standard_normal((4, 5, 6))
    gh = po.forward_axis(g, 1, N)
    for k in range(4):
        for i in range(6):
            np.testing.assert_allclose(gh[k, :, i], eq7(g[k, :, i]), rtol=0, atol=1e-13)
    gh = po.forward_axis(g, 2, D)
    np.testing.assert_allclose(gh[2, 3, :], eq9(g[2, 3, :]), rtol=0, atol=1e-13)


# ------------------------------------------------------------------ the paper's recipes
def read_examples():
    out = {}
    with open(os.path.join(GOLDEN, "paper_permutation_examples.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            name, src, dst, _ = [s.strip() for s in line.split("|")]
            out[name] = (src.split(), dst.split())
    return out


def symbolic(tokens, values):
    res = []
    for t in tokens:
        sign = -1.0 if t.startswith("-") else 1.0
        res.append(sign * values[int(t.lstrip("-u")) - 1])
    return np.array(res)


def test_paper_worked_examples():
    ex = read_examples()
    vals = np.array([1.5, -2.0, 3.25, 4.0, -5.5])
    src, dst = ex["makhoul_permute"]
    np.testing.assert_array_equal(mk.makhoul_permute(symbolic(src, vals)), symbolic(dst, vals))
    np.testing.assert_array_equal(mk.makhoul_unpermute(symbolic(dst, vals)), symbolic(src, vals))
    src, dst = ex["reverse_alternate"]
    np.testing.assert_array_equal(mk.reverse_alternate(symbolic(src, vals)), symbolic(dst, vals))


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 8, 9, 16, 31, 64])
def test_makhoul_recipes_equal_the_definitions(n):
    rng = np.random.default_rng(200 + n)
    u = rng.standard_normal(n)
    np.testing.assert_allclose(mk.dct10(u), eq7(u), rtol=0, atol=1e-12)
    np.testing.assert_allclose(mk.dst10(u), eq9(u), rtol=0, atol=1e-12)
    x, imag = mk.dct01(eq7(u))
    np.testing.assert_allclose(x, u, rtol=0, atol=1e-12)
    assert imag < 1e-12
    x, imag = mk.dst01(eq9(u))
    np.testing.assert_allclose(x, u, rtol=0, atol=1e-12)
    assert imag < 1e-12
    Y = rng.standard_normal(n)
    np.testing.assert_allclose(mk.dct01(Y)[0], (2.0 / n) * eq8(Y), rtol=0, atol=1e-12)
    np.testing.assert_allclose(mk.dst01(Y)[0], (2.0 / n) * eq10(Y), rtol=0, atol=1e-12)


@pytest.mark.parametrize("n", [4, 5])
def test_rearranging_twice(n):
    """PAPER.md:186 says rearranging twice recovers the signal; it gives (-1)^(N-1) u (R7)."""
    u = np.arange(1.0, n + 1)
    np.testing.assert_array_equal(mk.reverse_alternate(mk.reverse_alternate(u)), (-1.0) ** (n - 1) * u)
