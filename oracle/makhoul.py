"""The paper's three-step recipes for the real transforms -- pre-process, complex FFT,
post-process -- written out step by step in the paper's order.

TEST INFRASTRUCTURE ONLY (see ``oracle/__init__.py``).  These functions exist to pin the
*readings* of the garbled passages (R4-R7): ``tests/test_oracle_transforms.py``
checks each against the literal sums of eq. 7-10 and against the paper's two worked
5-element examples.  ``numpy.fft`` is the "complex FFT"
library step.  1-D, real input, any length N >= 1.
"""
from __future__ import annotations

import numpy as np


def makhoul_permute(u):
    """"take the even points in order then append the odd points in reverse
    order" -- ``[u1,u2,u3,u4,u5] -> [u1,u3,u5,u4,u2]``:  v_n = u_{2n},  v_{N-1-n} = u_{2n+1}."""
    u = np.asarray(u)
    return np.concatenate([u[0::2], u[1::2][::-1]])


def makhoul_unpermute(v):
    """Inverse of :func:`makhoul_permute` ("Retrieve the data assuming that it has been
    previously rearranged by a DCT10 transform")."""
    v = np.asarray(v)
    n = v.shape[0]
    u = np.empty_like(v)
    ne = (n + 1) // 2
    u[0::2] = v[:ne]
    u[1::2] = v[ne:][::-1]
    return u


def dct10(u):
    """DCT-II, eq. 7, by PAPER.md:131-146:
    permute -> complex FFT -> (Hermitian symmetry: the input is real, so only V_k is needed,
    R4) -> scale by exp(-sqrt(-1) k pi / 2N) -> keep the real part.  R3: eq. 7 carries no
    factor 2, so none is applied here."""
    u = np.asarray(u, dtype=np.float64)
    n = u.shape[0]
    V = np.fft.fft(makhoul_permute(u))
    k = np.arange(n)
    return np.real(np.exp(-1j * np.pi * k / (2 * n)) * V)


def dct01(Y):
    """The inverse of :func:`dct10`, PAPER.md:155-159 with R5 for the garbled first step:
    V_k = exp(+sqrt(-1) k pi / 2N) (Y_k - sqrt(-1) Y_{N-k}),  Y_N := 0;  v = IFFT(V) (1/N);
    un-permute.  Equals (2/N) x eq. 8 (DCT-III)."""
    Y = np.asarray(Y, dtype=np.float64)
    n = Y.shape[0]
    k = np.arange(n)
    Yrev = np.concatenate([[0.0], Y[:0:-1]])  # Y_{N-k}, with Y_N = 0 at k = 0
    V = np.exp(1j * np.pi * k / (2 * n)) * (Y - 1j * Yrev)
    v = np.fft.ifft(V)
    return makhoul_unpermute(v.real), float(np.max(np.abs(v.imag))) if n else 0.0


def reverse_alternate(u):
    """PAPER.md:170 / 172 / 181 / 184: ``[u1,u2,u3,u4,u5] -> [u5,-u4,u3,-u2,u1]``, i.e.
    out_m = (-1)^m u_{N-1-m}."""
    u = np.asarray(u)
    n = u.shape[0]
    sign = np.where(np.arange(n) % 2 == 0, 1.0, -1.0)
    return sign * u[::-1]


def dst10(u):
    """DST-II, eq. 9: rearrange, DCT10, rearrange (R7)."""
    return reverse_alternate(dct10(reverse_alternate(u)))


def dst01(Y):
    """The inverse of :func:`dst10`: rearrange, DCT01, rearrange.
    Equals (2/N) x the corrected eq. 10 (DST-III, R6)."""
    x, imag = dct01(reverse_alternate(Y))
    return reverse_alternate(x), imag
