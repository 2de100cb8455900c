"""Pins for the oracle's 1-D sweep and its multi-dimensional application
(p5-p9, layout and sign pins).  CPU only; never calls the CUDA path."""
import math

import numpy as np
import pytest

from oracle import oracle as O


def roll_cells(u, k, s):
    """exact permutation: cell i of the result is cell i-s of u."""
    n = k + 1
    return np.roll(u.reshape(-1, n), s, axis=0).reshape(-1)


@pytest.mark.parametrize("k", [0, 1, 2, 3])
@pytest.mark.parametrize("s", [0, 1, -1, 3, -3, 9, -10, 23])
def test_p5_integer_shift_is_exact_permutation(k, s):
    N = 7
    rng = np.random.default_rng(5)
    u = rng.standard_normal(N * (k + 1))
    u[3] = -0.0                                   # sign of zero must survive (pure copy)
    got = O.sweep_line(k, u, float(s))
    want = roll_cells(u, k, s)
    assert got.tobytes() == want.tobytes()


@pytest.mark.parametrize("k", [1, 2, 3])
@pytest.mark.parametrize("delta", [0.3, -0.3, 1.6, -2.2])
def test_p6_polynomial_of_degree_k_is_translated_exactly(k, delta):
    N = 12
    xi, _ = O.gauss_legendre(k + 1)
    y = (np.arange(N)[:, None] + xi[None, :]).reshape(-1)       # node positions in cell units
    rng = np.random.default_rng(k)
    c = rng.uniform(-1, 1, k + 1)
    p = lambda t: sum(cm * (t / N) ** m for m, cm in enumerate(c))
    got = O.sweep_line(k, p(y), delta)
    want = p(y - delta)
    # cells whose two donors do not wrap around the periodic boundary
    s = math.floor(delta)
    ok = np.array([(0 <= i - s - 1) and (i - s <= N - 1) for i in range(N)])
    mask = np.repeat(ok, k + 1)
    assert mask.sum() >= (N - 5) * (k + 1)
    assert np.abs(got - want)[mask].max() < 5e-15


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_p7_mass_and_constants_preserved_by_a_sweep(k):
    N = 9
    _, w = O.gauss_legendre(k + 1)
    rng = np.random.default_rng(11)
    u = rng.uniform(0, 1, N * (k + 1))
    W = np.tile(w, N)
    for delta in (0.37, -0.81, 4.25, -13.5):
        v = O.sweep_line(k, u, delta)
        assert abs((W * v).sum() - (W * u).sum()) < 1e-13
        c = O.sweep_line(k, np.full_like(u, 2.5), delta)
        assert np.abs(c - 2.5).max() < 1e-14


@pytest.mark.parametrize("k", [1, 2, 3])
def test_p8_order_of_convergence_is_k_plus_1(k):
    """advect sin(2 pi y) by M steps of 0.3 cells (a genuine projection each; alpha = 0.5 would be
    super-convergent for odd k by symmetry) and compare
    with the exact translate: error ~ h^(k+1) (PAPER.md:108 'The resulting numerical scheme has
    order k+1')."""
    xi, w = O.gauss_legendre(k + 1)
    errs = []
    M = 8
    for N in (8, 16, 32):
        y = (np.arange(N)[:, None] + xi[None, :]).reshape(-1) / N
        u = np.sin(2 * np.pi * y)
        for _ in range(M):
            u = O.sweep_line(k, u, 0.3)
        exact = np.sin(2 * np.pi * (y - M * 0.3 / N))
        errs.append(np.sqrt((np.tile(w, N) * (u - exact) ** 2).sum() / N))
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert 2 ** (k + 1) * 0.85 < r1 < 2 ** (k + 1) * 1.2
    assert 2 ** (k + 1) * 0.9 < r2 < 2 ** (k + 1) * 1.1


def test_full_period_in_integer_steps_returns_initial_data_exactly():
    k, N = 2, 10
    rng = np.random.default_rng(2)
    u0 = rng.standard_normal(N * (k + 1))
    u = u0.copy()
    for _ in range(5):
        u = O.sweep_line(k, u, 2.0)
    assert u.tobytes() == u0.tobytes()


@pytest.mark.parametrize("k", [1, 2])
def test_p9_locality_two_adjacent_cells(k):
    N, n = 11, k + 1
    rng = np.random.default_rng(3)
    u = rng.standard_normal(N * n)
    for delta in (0.4, -0.4, 2.7, -5.1):
        base = O.sweep_line(k, u, delta)
        v = u.copy()
        v[4 * n: 5 * n] += 1.0                      # perturb input cell 4
        diff = np.abs(O.sweep_line(k, v, delta) - base).reshape(N, n).max(axis=1) > 0
        s = math.floor(delta)
        # input cell m feeds output cells m+s (via A) and m+s+1 (via B)
        assert set(np.nonzero(diff)[0]) == {(4 + s) % N, (4 + s + 1) % N}


# --------------------------------------------------------------- multi-dimensional application

def make(dx, dv, cells, k, dom=None):
    if dom is None:
        dom = []
        for a in range(dx + dv):
            dom += [0.0, 1.0 + a] if a < dx else [-2.0 - a, 2.0 + a]
    return O.Oracle(dx, dv, cells, k, dom)


def test_sweep_axis_layout_against_numpy_line_by_line():
    """x_1 fastest; numpy shape (D_last..D_0).  Every line along `axis` must equal sweep_line on that
    line with the delta of its shift index (x-sweep: node of v-axis dx+axis; v-sweep: flat x node)."""
    orc = make(2, 2, [3, 4, 2, 3], 1)
    rng = np.random.default_rng(8)
    f = rng.uniform(0, 1, orc.shape)
    D = orc.D
    for axis in range(4):
        if axis < 2:
            delta = rng.uniform(-2.5, 2.5, D[2 + axis])
        else:
            delta = rng.uniform(-2.5, 2.5, orc.X)
        got = orc.sweep_axis(f, axis, delta)
        want = np.empty_like(f)
        g = np.moveaxis(f, 3 - axis, -1)              # numpy axis of phase-space axis a is 3-a
        wv = np.moveaxis(want, 3 - axis, -1)
        it = np.ndindex(*g.shape[:-1])
        other = [a for a in range(4) if a != axis]    # phase axes of g's leading dims, reversed order
        lead_axes = [a for a in reversed(range(4)) if a != axis]
        for idx in it:
            node = dict(zip(lead_axes, idx))
            if axis < 2:
                dlt = delta[node[2 + axis]]
            else:
                dlt = delta[node[0] + D[0] * node[1]]
            wv[idx] = O.sweep_line(1, np.ascontiguousarray(g[idx]), dlt)
        assert np.array_equal(got, want)


def test_advect_x_moves_a_linear_profile_by_v_tau():
    """f(x,v) = x_1  ->  f(x_1 - v_1 tau)  (step 1a); pins the sign and the v-node lookup."""
    orc = make(1, 1, [16, 6], 1, [0.0, 8.0, -3.0, 3.0])
    x, v = orc.node_coords(0), orc.node_coords(1)
    f = np.broadcast_to(x[None, :], orc.shape).copy()
    tau = 0.37
    g = orc.advect_x(f, tau)
    want = x[None, :] - v[:, None] * tau
    h = 0.5
    interior = (x > 2 * h + 3 * tau) & (x < 8 - 2 * h - 3 * tau)
    assert np.abs(g - want)[:, interior].max() < 1e-13


def test_advect_v_moves_a_linear_profile_by_plus_E_tau():
    """f(x,v) = v_1 -> f(x, v_1 + E_1(x) tau) = v_1 + E_1 tau (step 3a; sign of eq. (1))."""
    orc = make(1, 1, [5, 16], 1, [0.0, 1.0, -4.0, 4.0])
    x, v = orc.node_coords(0), orc.node_coords(1)
    f = np.broadcast_to(v[:, None], orc.shape).copy()
    E = np.linspace(-0.9, 1.1, orc.X)
    tau = 0.6
    g = orc.advect_v(f, E, tau)
    want = v[:, None] + E[None, :] * tau
    interior = np.abs(v) < 4 - 2 * 0.5 - 1.1 * tau
    assert np.abs(g - want)[interior, :].max() < 1e-13


def test_advect_x_2x3v_and_3x3v_use_matching_velocity_axis_and_leave_others():
    """x_d is moved by v_d (steps 1a-1c); with integer shifts the result is an exact roll per v-node."""
    for dx, dv in ((2, 3), (3, 3)):
        d = dx + dv
        cells = [4, 3, 5, 2, 3, 2][:d] if dx == 3 else [4, 3, 2, 3, 2]
        k = 0                                        # k=0: nodes at cell centres -> integer delta by choice of domain
        dom = []
        for a in range(d):
            if a < dx:
                dom += [0.0, float(cells[a])]        # h_x = 1
            else:
                dom += [0.0, float(cells[a])]        # v nodes at 0.5, 1.5, ...
        orc = O.Oracle(dx, dv, cells, k, dom)
        rng = np.random.default_rng(dx)
        f = rng.uniform(0, 1, orc.shape)
        tau = 2.0                                     # delta = v*tau/h = 1, 3, 5, ...
        got = orc.advect_x(f, tau)
        want = f.copy()
        for a in range(dx):
            va = orc.node_coords(dx + a)
            npax_x, npax_v = d - 1 - a, d - 1 - (dx + a)
            tmp = np.empty_like(want)
            for n, vv in enumerate(va):
                sl = [slice(None)] * d
                sl[npax_v] = n
                tmp[tuple(sl)] = np.roll(want[tuple(sl)], int(round(vv * tau)), axis=npax_x - (1 if npax_v < npax_x else 0))
            want = tmp
        assert np.array_equal(got, want)


def test_advect_v_2x3v_leaves_v3_untouched_and_uses_minus_E():
    cells = [2, 3, 4, 5, 3]
    dom = [0, 2.0, 0, 3.0, 0, 4.0, 0, 5.0, 0, 3.0]    # all h = 1
    orc = O.Oracle(2, 3, cells, 0, dom)
    rng = np.random.default_rng(4)
    f = rng.uniform(0, 1, orc.shape)
    E = np.zeros((2,) + orc.xshape)
    E[0] = rng.integers(-2, 3, orc.xshape)
    E[1] = rng.integers(-2, 3, orc.xshape)
    got = orc.advect_v(f, E, 1.0)                     # delta = -E exactly
    want = np.empty_like(f)
    # f_new(x, v) = f(x, v + E): cell i takes cell i+E -> roll by -E along v_1 then v_2
    for ix2 in range(3):
        for ix1 in range(2):
            blk = f[:, :, :, ix2, ix1]
            blk = np.roll(blk, -int(E[0, ix2, ix1]), axis=2)      # v_1 is numpy axis 2 of (v3,v2,v1)
            blk = np.roll(blk, -int(E[1, ix2, ix1]), axis=1)      # v_2
            want[:, :, :, ix2, ix1] = blk
    assert np.array_equal(got, want)


def test_x_sweeps_commute_to_roundoff():
    """'no error is introduced by this splitting as the corresponding operators commute'."""
    orc = make(2, 2, [5, 4, 3, 3], 2)
    rng = np.random.default_rng(9)
    f = rng.uniform(0, 1, orc.shape)
    d0 = rng.uniform(-1.5, 1.5, orc.D[2])
    d1 = rng.uniform(-1.5, 1.5, orc.D[3])
    a = orc.sweep_axis(orc.sweep_axis(f, 0, d0), 1, d1)
    b = orc.sweep_axis(orc.sweep_axis(f, 1, d1), 0, d0)
    assert np.abs(a - b).max() < 1e-14


def test_mass_conserved_by_every_sweep_and_by_strang_steps():
    orc = make(2, 2, [4, 4, 6, 6], 2, [0, 4 * np.pi, 0, 4 * np.pi, -6, 6, -6, 6])
    rng = np.random.default_rng(10)
    x1, x2, v1, v2 = (orc.node_coords(a) for a in range(4))
    f = (np.exp(-0.5 * (v1[None, :, None, None] ** 2 + v2[:, None, None, None] ** 2)) / (2 * np.pi)
         * (1 + 0.05 * np.cos(0.5 * x1)[None, None, None, :] + 0.05 * np.cos(0.5 * x2)[None, None, :, None]))
    f = f * (1 + 1e-3 * rng.uniform(-1, 1, f.shape))
    m0 = orc.mass(f)
    for _ in range(5):
        f, rho, E = orc.step(f, 0.1)
    assert abs(orc.mass(f) - m0) < 2e-14 * abs(m0) * 10
