"""CPU checks of the PRODUCT's host logic (no GPU, no compute kernels): the Gauss-Legendre rule and the
A(alpha), B(alpha) tables of libsldg_b200.so, in both arithmetic routes --

  device_arith = 0: long-double Horner on the host (x-sweep tables),
  device_arith = 1: the fp64 fused-multiply-add Horner of the device-side v-sweep table kernel, reproduced on the
                    host by sldg_AB (same coefficients, same operation order) --

against what the mathematics fixes (numpy's leggauss, the k = 0 and k = 1 closed forms p1/p2, the printed values
p3, the invariants p4) and against the independently written oracle (different route: quadrature of the
definition; the product expands the Lagrange basis and integrates in closed form).
"""
import math
import os

import numpy as np
import pytest

import paper_2110_14557_b200 as P
from oracle import oracle as O

S3 = math.sqrt(3.0)
ROUTES = [0, 1]


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_gauss_legendre_matches_numpy(k):
    xi, w = P.gauss_legendre(k)
    t, wt = np.polynomial.legendre.leggauss(k + 1)
    assert np.abs(xi - (t + 1) / 2).max() <= 4 * 2.3e-16
    assert np.abs(w - wt / 2).max() <= 4 * 2.3e-16
    assert abs(w.sum() - 1) < 1e-15


@pytest.mark.parametrize("route", ROUTES)
def test_k0_upwind_and_k1_closed_form(route):
    for a in (0.0, 1e-9, 0.123, 0.3, 0.5, 0.77, 1 - 1e-9, 1.0):
        A, B = P.AB(0, a, route)
        assert abs(A[0, 0] - (1 - a)) < 3e-16 and abs(B[0, 0] - a) < 3e-16
        A, B = P.AB(1, a, route)
        Ar = np.array([[1 - 2 * a + a**3, (1 - S3) * a + S3 * a**2 - a**3],
                       [(1 + S3) * a - S3 * a**2 - a**3, 1 - 2 * a + a**3]])
        Br = np.array([[-a + 3 * a**2 - a**3, (2 + S3) * a - (3 + S3) * a**2 + a**3],
                       [(2 - S3) * a - (3 - S3) * a**2 + a**3, -a + 3 * a**2 - a**3]])
        assert np.abs(A - Ar).max() < 2e-15 and np.abs(B - Br).max() < 2e-15


@pytest.mark.parametrize("route", ROUTES)
def test_printed_values_alpha_0p3(golden_dir, route):
    want = {}
    with open(os.path.join(golden_dir, "ab_alpha0p3.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            tok = line.split()
            want[(int(tok[0]), tok[1], int(tok[2]))] = [float(t) for t in tok[3:]]
    for k in (1, 2):
        A, B = P.AB(k, 0.3, route)
        for j in range(k + 1):
            assert np.abs(A[j] - want[(k, "A", j)]).max() < 2e-15
            assert np.abs(B[j] - want[(k, "B", j)]).max() < 2e-15


@pytest.mark.parametrize("route", ROUTES)
@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_invariants_and_oracle_agreement(k, route):
    n = k + 1
    xi, w = P.gauss_legendre(k)
    A0, B0 = P.AB(k, 0.0, route)
    A1, B1 = P.AB(k, 1.0, route)
    tol = 1e-14
    assert np.abs(A0 - np.eye(n)).max() < tol and np.abs(B0).max() < tol
    assert np.abs(A1).max() < tol and np.abs(B1 - np.eye(n)).max() < tol
    alphas = list(np.linspace(0, 1, 101)) + [1e-12, 1e-6, 1e-3, 0.999, 1 - 1e-6, 1 - 1e-12]
    worst = 0.0
    for a in alphas:
        A, B = P.AB(k, a, route)
        assert np.abs((A + B).sum(axis=1) - 1).max() < 2e-14            # constants preserved
        assert np.abs(w @ (A + B) - w).max() < 1e-14                    # mass
        Ar, _ = P.AB(k, 1.0 - a, route)
        assert np.abs(B - Ar[::-1, ::-1]).max() < 2e-14                 # reflection
        Ao, Bo = O.AB(k, a)
        worst = max(worst, np.abs(A - Ao).max(), np.abs(B - Bo).max())
    # both are fp64-rounded evaluations of the same polynomial; the bound that the 1e-12 sweep parity needs is
    # far looser
    assert worst < 5e-15, worst


def test_argument_validation():
    L = P.lib()
    import ctypes as C
    a = (C.c_double * 25)()
    assert L.sldg_AB(5, 0.5, 0, a, a) == -1
    assert L.sldg_AB(1, 1.5, 0, a, a) == -1
    assert L.sldg_AB(1, float("nan"), 0, a, a) == -1
    assert L.sldg_AB(1, 0.5, 0, None, a) == -1
    assert L.sldg_gauss_legendre(-1, a, a) == -1


@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_sipg_matrices_host(k):
    """M, B of the CGdG solver (reading I) as the library builds them on the host: against the
    independently written oracle, and the properties eq. (4) fixes -- M symmetric, rows of M + B + B^T sum to 0
    (constants are in the null space)."""
    M, B = P.sipg_matrices(k)
    Mo, Bo = O.sipg_MB(k, O.sipg_sigma_default(k))
    assert np.abs(M - Mo).max() < 1e-12 * np.abs(Mo).max() and np.abs(B - Bo).max() < 1e-12 * np.abs(Mo).max()
    assert np.abs(M - M.T).max() < 1e-13 * np.abs(M).max()
    assert np.abs((M + B + B.T).sum(axis=1)).max() < 1e-12 * np.abs(M).max()
    assert P.lib().sldg_sipg_matrices(0, 1.0, M.ctypes.data_as(P.binding._dp), B.ctypes.data_as(P.binding._dp)) == -1
