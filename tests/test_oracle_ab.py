"""Pins for the oracle's constants and A(alpha), B(alpha) (pins p1-p4, p13).

Nothing here calls the CUDA path.  Independent references: numpy's leggauss, closed forms,
mpmath quadrature of the translate-then-L2-project definition (Fig. 1).
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

from oracle import oracle as O

S3 = math.sqrt(3.0)


def np_gl01(n):
    t, w = np.polynomial.legendre.leggauss(n)
    return (t + 1) / 2, w / 2


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6])
def test_gauss_legendre_matches_numpy_and_textbook(n):
    xi, w = O.gauss_legendre(n)
    xr, wr = np_gl01(n)
    assert np.allclose(xi, xr, rtol=0, atol=2e-16 * 4)
    assert np.allclose(w, wr, rtol=0, atol=2e-16 * 4)
    assert abs(w.sum() - 1) < 1e-15
    if n == 2:   # textbook: 1/2 -+ sqrt(3)/6
        assert np.allclose(xi, [0.5 - S3 / 6, 0.5 + S3 / 6], atol=1e-16)
    if n == 3:   # textbook: 1/2 -+ sqrt(15)/10, weights 5/18 4/9 5/18
        assert np.allclose(xi, [0.5 - math.sqrt(15) / 10, 0.5, 0.5 + math.sqrt(15) / 10], atol=1e-16)
        assert np.allclose(w, [5 / 18, 4 / 9, 5 / 18], atol=1e-16)


def test_lagrange_is_cardinal_and_partition_of_unity():
    for n in (2, 3, 4, 5):
        xi, _ = O.gauss_legendre(n)
        for l in range(n):
            for q in range(n):
                assert O.lagrange(xi, l, xi[q]) == (1.0 if l == q else 0.0)
        for z in (-0.3, 0.0, 0.37, 1.0, 1.4):
            assert abs(sum(O.lagrange(xi, l, z) for l in range(n)) - 1) < 1e-13


def test_p1_k0_is_first_order_upwind():
    for a in (0.0, 0.1, 0.5, 0.999):
        A, B = O.AB(0, a)
        assert abs(A[0, 0] - (1 - a)) < 1e-16 and abs(B[0, 0] - a) < 1e-16


def test_p2_k1_closed_form():
    for a in (0.0, 1e-9, 0.123, 0.3, 0.5, 0.77, 1 - 1e-9):
        A, B = O.AB(1, a)
        Ar = np.array([[1 - 2 * a + a**3, (1 - S3) * a + S3 * a**2 - a**3],
                       [(1 + S3) * a - S3 * a**2 - a**3, 1 - 2 * a + a**3]])
        Br = np.array([[-a + 3 * a**2 - a**3, (2 + S3) * a - (3 + S3) * a**2 + a**3],
                       [(2 - S3) * a - (3 - S3) * a**2 + a**3, -a + 3 * a**2 - a**3]])
        assert np.abs(A - Ar).max() < 2e-15
        assert np.abs(B - Br).max() < 2e-15


def test_p3_printed_values(golden_dir):
    want = {}
    with open(os.path.join(golden_dir, "ab_alpha0p3.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            tok = line.split()
            want[(int(tok[0]), tok[1], int(tok[2]))] = [float(t) for t in tok[3:]]
    for k in (1, 2):
        A, B = O.AB(k, 0.3)
        for j in range(k + 1):
            assert np.abs(A[j] - want[(k, "A", j)]).max() < 2e-16 * 8
            assert np.abs(B[j] - want[(k, "B", j)]).max() < 2e-16 * 8


def mp_AB(k, alpha, dps=30):
    """A, B from the definition with mpmath: project the translated basis function.
    A_jl = (1/w_j) int_alpha^1 l_j(x) l_l(x-alpha) dx ; B_jl = (1/w_j) int_0^alpha l_j(x) l_l(x-alpha+1) dx,
    nodes/weights from mpmath's own Legendre roots."""
    mp.mp.dps = dps
    n = k + 1
    roots = sorted(mp.polyroots([mp.mpf(c) for c in np.polynomial.legendre.leg2poly([0] * n + [1])[::-1]],
                                maxsteps=200, extraprec=200))
    xi = [(r + 1) / 2 for r in roots]

    def lag(l, z):
        r = mp.mpf(1)
        for m in range(n):
            if m != l:
                r *= (z - xi[m]) / (xi[l] - xi[m])
        return r
    w = [mp.quad(lambda z, l=l: lag(l, z), [0, 1]) for l in range(n)]
    a = mp.mpf(alpha)
    A = np.zeros((n, n)); B = np.zeros((n, n))
    for j in range(n):
        for l in range(n):
            A[j, l] = float(mp.quad(lambda z: lag(j, z) * lag(l, z - a), [a, 1]) / w[j])
            B[j, l] = float(mp.quad(lambda z: lag(j, z) * lag(l, z - a + 1), [0, a]) / w[j])
    return A, B


@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_AB_against_mpmath_definition(k):
    for alpha in (0.3, 0.8125):
        A, B = O.AB(k, alpha)
        Ar, Br = mp_AB(k, alpha)
        assert np.abs(A - Ar).max() < 1e-14
        assert np.abs(B - Br).max() < 1e-14


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_p4_invariants(k):
    n = k + 1
    xi, w = O.gauss_legendre(n)
    A0, B0 = O.AB(k, 0.0)
    assert np.array_equal(A0, np.eye(n)) or np.abs(A0 - np.eye(n)).max() < 1e-15
    assert np.abs(B0).max() == 0.0
    A1, B1 = O.AB(k, 1.0 - 1e-15)
    assert np.abs(A1).max() < 1e-13 and np.abs(B1 - np.eye(n)).max() < 1e-13
    rng = np.random.default_rng(7)
    for alpha in rng.uniform(0, 1, 6):
        A, B = O.AB(k, alpha)
        # constants preserved
        assert np.abs((A + B).sum(axis=1) - 1).max() < 1e-13
        # mass: sum_j w_j (A+B)_jl = w_l
        assert np.abs(w @ (A + B) - w).max() < 1e-14
        # reflection symmetry B_jl(alpha) = A_{k-j,k-l}(1-alpha)
        Ar, _ = O.AB(k, 1.0 - alpha)
        assert np.abs(B - Ar[::-1, ::-1]).max() < 1e-13
    # every entry is a polynomial of degree <= 2k+1 in alpha: a degree-(2k+1) fit through 2k+2
    # Chebyshev points reproduces other points
    m = 2 * k + 2
    pts = 0.5 - 0.5 * np.cos((np.arange(m) + 0.5) * np.pi / m)
    vals = np.array([np.concatenate([M.ravel() for M in O.AB(k, a)]) for a in pts])
    coef = np.polynomial.polynomial.polyfit(pts, vals, m - 1)
    for a in (0.05, 0.41, 0.93):
        got = np.concatenate([M.ravel() for M in O.AB(k, a)])
        assert np.abs(np.polynomial.polynomial.polyval(a, coef) - got).max() < 1e-11


def brute_force_sweep(k, u, delta, dps=25):
    """p13: translate the piecewise polynomial by delta cells and L2-project, cell by cell, with
    mpmath quadrature split at the discontinuity.  No A/B, no donor bookkeeping."""
    mp.mp.dps = dps
    n = k + 1
    xi, w = np_gl01(n)
    N = len(u) // n

    def lag(l, z):
        r = mp.mpf(1)
        for m in range(n):
            if m != l:
                r *= (z - mp.mpf(xi[m])) / (mp.mpf(xi[l]) - mp.mpf(xi[m]))
        return r

    def U(y):                      # periodic piecewise polynomial, y in cell units
        c = int(mp.floor(y))
        z = y - c
        c %= N
        return sum(mp.mpf(float(u[c * n + l])) * lag(l, z) for l in range(n))
    out = np.zeros_like(u)
    brk = float(delta - math.floor(delta))
    for i in range(N):
        for j in range(n):
            pts = [0, brk, 1] if 0 < brk < 1 else [0, 1]
            val = mp.quad(lambda z: lag(j, z) * U(i + z - mp.mpf(delta)), pts)
            out[i * n + j] = float(val / mp.mpf(w[j]))
    return out


@pytest.mark.parametrize("k,N,delta", [(0, 4, 0.3), (1, 3, 0.3), (1, 4, -0.45), (2, 3, 1.7),
                                       (2, 5, -2.25), (3, 3, 0.6), (1, 3, 4.5), (2, 4, -7.75)])
def test_p13_sweep_line_against_brute_force_projection(k, N, delta):
    rng = np.random.default_rng(100 * k + N)
    u = rng.uniform(-1, 1, N * (k + 1))
    got = O.sweep_line(k, u, delta)
    want = brute_force_sweep(k, u, delta)
    assert np.abs(got - want).max() < 1e-13
