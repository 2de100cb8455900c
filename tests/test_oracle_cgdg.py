"""Pins for the oracle's CGdG Poisson solver (SIPG discretisation + mean-preserving CG, PAPER.md:496-567,
SURVEY 8(f) rank 3; readings I, T, U, V of DESIGN.md section 3.2).

Nothing here calls the CUDA path.  Independent references: the bilinear form of eq. (4) evaluated
directly on numpy polynomials (derivatives, integrals, jumps and averages by numpy.polynomial, no M/B matrices),
numpy.linalg (eigvalsh, lstsq) on the dense matrix, closed-form solutions, and the oracle's
own FFT-route solver, which is pinned separately.
"""
import numpy as np
import pytest
from numpy.polynomial import polynomial as Pn

from oracle import oracle as O


def ctx1d(N, k, L=4 * np.pi):
    return O.Oracle(1, 1, [N, 1], k, [0.0, L, -1.0, 1.0])


def dense(orc, sigma=None):
    X = orc.X
    A = np.empty((X, X))
    e = np.zeros(X)
    for j in range(X):
        e[j] = 1.0
        A[:, j] = orc.sipg_apply(e, sigma).reshape(-1)
        e[j] = 0.0
    return A


def cell_polys(orc, u):
    """numpy polynomials (in the reference coordinate z of each cell) through the nodal values of a 1-D vector"""
    k = orc.k
    xi, _ = O.gauss_legendre(k + 1)
    return [Pn.Polynomial(Pn.polyfit(xi, u[i * (k + 1):(i + 1) * (k + 1)], k)) for i in range(orc.cells[0])]


def bilinear_eq4(orc, u, v, sigma):
    """a(u, v) of eq. (4) for periodic 1-D piecewise polynomials, straight from its definition:
    sum_i int_{I_i} u' v' - sum_faces ({u'}[v] + {v'}[u]) + sigma/h sum_faces [u][v],
    [g] = g(x^-) - g(x^+), {g} = (g(x^-) + g(x^+))/2; physical derivative = (1/h) d/dz."""
    N, h = orc.cells[0], (orc.domain[1] - orc.domain[0]) / orc.cells[0]
    pu, pv = cell_polys(orc, u), cell_polys(orc, v)
    total = 0.0
    for i in range(N):
        integrand = (pu[i].deriv() * pv[i].deriv()).integ()
        total += (integrand(1.0) - integrand(0.0)) / h
        # face at the left end of cell i: minus side = right end of cell i-1, plus side = left end of cell i
        um, up, vm, vp = pu[i - 1](1.0), pu[i](0.0), pv[i - 1](1.0), pv[i](0.0)
        dum, dup = pu[i - 1].deriv()(1.0) / h, pu[i].deriv()(0.0) / h
        dvm, dvp = pv[i - 1].deriv()(1.0) / h, pv[i].deriv()(0.0) / h
        total -= 0.5 * (dum + dup) * (vm - vp) + 0.5 * (dvm + dvp) * (um - up)
        total += sigma / h * (um - up) * (vm - vp)
    return total


# --------------------------------------------------------------- basis derivative

@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_lagrange_derivative_matches_numpy_polynomial(k):
    xi, _ = O.gauss_legendre(k + 1)
    for l in range(k + 1):
        e = np.zeros(k + 1); e[l] = 1.0
        p = Pn.Polynomial(Pn.polyfit(xi, e, k)).deriv()
        for z in (0.0, 0.3, 1.0, *xi):
            assert abs(O.lagrange_deriv(xi, l, z) - p(z)) < 1e-10 * (1 + abs(p(z)))


# --------------------------------------------------------------- the operator against eq. (4) itself

@pytest.mark.parametrize("k,N", [(1, 5), (2, 4), (3, 3), (4, 3)])
@pytest.mark.parametrize("sigma", [None, 7.5])
def test_operator_is_the_bilinear_form_of_eq4(k, N, sigma):
    """v^T (A u) == a(u, v) evaluated from the definition on random piecewise polynomials: pins M, B, their
    placement (B couples cell i-1, B^T cell i+1), the 1/h scaling and the signs of every flux term."""
    orc = ctx1d(N, k, L=3.0)
    s = O.sipg_sigma_default(k) if sigma is None else sigma
    rng = np.random.default_rng(7 + k)
    for _ in range(4):
        u, v = rng.standard_normal(orc.X), rng.standard_normal(orc.X)
        got = float(v @ orc.sipg_apply(u, s).reshape(-1))
        want = bilinear_eq4(orc, u, v, s)
        assert abs(got - want) < 1e-10 * (abs(want) + np.abs(u).max() * np.abs(v).max() * N)


@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_operator_is_symmetric_semidefinite_with_constant_null_vector(k):
    """symmetric, positive (semi)definite for sigma at its minimum allowed value; the only null
    vector is the constant.  Reading T: for k = 1, sigma = k^2 = 1 has a second null vector."""
    orc = ctx1d(8, k)
    A = dense(orc)
    assert np.abs(A - A.T).max() < 1e-12 * np.abs(A).max()
    assert np.abs(A @ np.ones(orc.X)).max() < 1e-12 * np.abs(A).max()
    ev = np.linalg.eigvalsh((A + A.T) / 2)
    assert ev[0] > -1e-12 * ev[-1] and ev[1] > 1e-3 * ev[-1] / orc.X ** 2
    if k == 1:
        ev1 = np.linalg.eigvalsh(dense(orc, sigma=1.0))
        assert abs(ev1[1]) < 1e-12 * ev1[-1]


def test_tensor_product_form_in_2d():
    """(h_y W_y (x) A_x + h_x A_y (x) W_x) u = b, checked against the two 1-D operators."""
    k, Nx, Ny, Lx, Ly = 2, 4, 3, 2.0, 3.0
    o2 = O.Oracle(2, 2, [Nx, Ny, 1, 1], k, [0, Lx, 0, Ly, -1, 1, -1, 1])
    ox, oy = ctx1d(Nx, k, Lx), ctx1d(Ny, k, Ly)
    Ax, Ay = dense(ox), dense(oy)
    _, w = O.gauss_legendre(k + 1)
    Wx, Wy = np.diag(np.tile(w, Nx)), np.diag(np.tile(w, Ny))
    A2 = (Ly / Ny) * np.kron(Wy, Ax) + (Lx / Nx) * np.kron(Ay, Wx)        # y is the slow index
    u = np.random.default_rng(3).standard_normal(o2.X)
    assert np.abs(o2.sipg_apply(u).reshape(-1) - A2 @ u).max() < 1e-12 * np.abs(A2).max() * np.abs(u).max()


# --------------------------------------------------------------- E = -grad phi (reading U)

def test_grad_phi_is_exact_for_polynomials_of_degree_k():
    k = 3
    orc = O.Oracle(2, 2, [3, 2, 1, 1], k, [0.0, 1.5, -1.0, 1.0, -1, 1, -1, 1])
    x, y = orc.node_coords(0), orc.node_coords(1)
    phi = (x ** 3 - 2 * x)[None, :] * (1 + y ** 2)[:, None]
    E = orc.grad_phi(phi)
    assert np.abs(E[0] + (3 * x ** 2 - 2)[None, :] * (1 + y ** 2)[:, None]).max() < 1e-12
    assert np.abs(E[1] + (x ** 3 - 2 * x)[None, :] * (2 * y)[:, None]).max() < 1e-12


# --------------------------------------------------------------- Algorithm 1

@pytest.mark.parametrize("dx,cells,k", [(1, [7], 2), (2, [5, 4], 1), (2, [4, 3], 3), (3, [3, 2, 3], 2)])
def test_cg_solution_is_the_mean_free_least_squares_solution(dx, cells, k):
    """Converged Algorithm 1 == numpy.linalg.lstsq on the dense matrix (minimum-norm = mean-free solution) with
    the mean of b removed (the system has no constraint on the mean)."""
    dom = []
    for a in range(dx):
        dom += [0.0, 2.0 + a]
    orc = O.Oracle(dx, dx, cells + [1] * dx, k, dom + [-1.0, 1.0] * dx)
    rng = np.random.default_rng(11)
    rho = 1.0 + 0.1 * rng.standard_normal(orc.xshape)
    E, phi, it, relres = orc.poisson_cg(rho, tol=1e-13, maxiter=2000)
    A = dense(orc)
    b = orc.sipg_rhs(rho).reshape(-1)
    want = np.linalg.lstsq(A, b - b.mean(), rcond=None)[0]
    assert relres < 1e-12
    assert abs(phi.mean()) < 1e-12 * np.abs(phi).max()
    assert np.abs(phi.reshape(-1) - want).max() < 1e-9 * np.abs(want).max()
    assert np.abs(E - orc.grad_phi(want)).max() < 1e-8 * np.abs(E).max()


@pytest.mark.parametrize("k", [1, 2, 3])
def test_cos_half_x_closed_form_converges_at_order_k_plus_1(k):
    """The paper's own check (figure 20): -phi'' = cos(0.5 x) periodic on [0,4pi] has
    phi = 4 cos(0.5 x); the error falls with order k+1."""
    errs = []
    for N in (8, 16, 32):
        orc = ctx1d(N, k)
        x = orc.node_coords(0)
        rho = 1.0 - np.cos(0.5 * x)
        _, phi, _, _ = orc.poisson_cg(rho, tol=1e-13, maxiter=5000)
        ex = 4 * np.cos(0.5 * x)
        errs.append(np.abs(phi - phi.mean() - (ex - ex.mean())).max() / 4)
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert orders[-1] > k + 1 - 0.35, (errs, orders)


def test_cgdg_field_agrees_with_the_fft_route_to_discretisation_error():
    """no significant difference between the FFT and the dG Poisson solver.  Landau density in 2-d:
    both fields approach -(eps/k) sin(k x_d); E from the dG potential is one order lower (derivative)."""
    k = 3
    orc = O.Oracle(2, 2, [8, 8, 1, 1], k, [0, 4 * np.pi, 0, 4 * np.pi, -1, 1, -1, 1])
    x, y = orc.node_coords(0), orc.node_coords(1)
    rho = 1 + 0.01 * (np.cos(0.5 * x)[None, :] + np.cos(0.5 * y)[:, None])
    Ecg, _, it, _ = orc.poisson_cg(rho, tol=1e-12, maxiter=2000)
    Efft = orc.poisson(rho)
    ex0 = -0.02 * np.sin(0.5 * x)[None, :] * np.ones_like(y)[:, None]
    assert np.abs(Efft[0] - ex0).max() < 2e-4 * 0.02
    assert np.abs(Ecg[0] - ex0).max() < 5e-3 * 0.02
    assert np.abs(Ecg - Efft).max() < 5e-3 * 0.02


def test_warm_start_and_iteration_bound():
    """starting from the previous potential needs few iterations; convergence within
    about (prod N_l (k_l+1))^(1/dx) iterations at the paper's tolerance 1e-3."""
    k = 2
    orc = O.Oracle(2, 2, [8, 8, 1, 1], k, [0, 4 * np.pi, 0, 4 * np.pi, -1, 1, -1, 1])
    x, y = orc.node_coords(0), orc.node_coords(1)
    rho = 1 + 0.01 * (np.cos(0.5 * x)[None, :] + np.cos(1.0 * y)[:, None] * np.sin(0.5 * x)[None, :])
    _, phi, it0, rel0 = orc.poisson_cg(rho, tol=1e-3)
    assert it0 <= round(orc.X ** 0.5) and rel0 < 1e-3
    _, phi1, it1, _ = orc.poisson_cg(rho, phi0=phi, tol=1e-3)
    assert it1 == 0 and np.array_equal(phi1, phi - phi.mean())          # already converged: untouched
    rho2 = rho + 1e-4 * np.cos(0.5 * x)[None, :]                         # "the next time step"
    _, _, it_cold, _ = orc.poisson_cg(rho2, tol=1e-5)
    _, _, it_warm, _ = orc.poisson_cg(rho2, phi0=phi, tol=1e-5)
    assert it_warm < it_cold


def test_cg_preserves_the_mean_with_an_inconsistent_right_hand_side():
    """Algorithm 1 removes the mean of r_0 and of A p: a density whose mean is not 1 (velocity
    truncation) still converges, the potential keeps mean 0, and the field equals that of rho - mean defect."""
    orc = O.Oracle(2, 2, [5, 4, 1, 1], 2, [0, 2.0, 0, 3.0, -1, 1, -1, 1])
    rng = np.random.default_rng(5)
    rho = 1.0 + 0.05 * rng.standard_normal(orc.xshape)
    b = orc.sipg_rhs(rho)
    W = orc.sipg_rhs(np.zeros(orc.xshape))                              # the weights W_x
    shift = b.mean() / W                                                # rho' = rho + shift makes sum(b') != 0 ...
    E1, phi1, _, r1 = orc.poisson_cg(rho, tol=1e-13, maxiter=3000)
    E2, phi2, _, r2 = orc.poisson_cg(rho + 0.3, tol=1e-13, maxiter=3000)
    assert abs(phi1.mean()) < 1e-13 * np.abs(phi1).max() and abs(phi2.mean()) < 1e-13 * np.abs(phi2).max()
    # a constant added to rho changes b by -0.3 W, whose projection off the constant vector is NOT zero unless the
    # weights are uniform; the solve must still converge (residual measured after mean removal)
    assert r1 < 1e-12 and r2 < 1e-10
