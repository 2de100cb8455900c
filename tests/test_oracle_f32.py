"""Pins for the oracle's single precision mode (Tables 3-4; reading W of
DESIGN.md: fp32 storage and sweep arithmetic, fp64 shift decisions, rho and field solve).

The fp64 oracle is pinned by tests/test_oracle_{ab,sweep,field}.py; the fp32 functions are the same statements
with float storage, pinned here by (a) closeness to the pinned fp64 result within the fp32 rounding bound of the
arithmetic, (b) what stays exact in any precision (integer shifts are bit-exact permutations), (c) conservation
to fp32 round-off, (d) the paper's statement that single and double precision results overlap.
"""
import numpy as np
import pytest

import workloads as W
from oracle import oracle as O

EPS32 = 2.0 ** -24


def rel_inf(a, b):
    return float(np.abs(a.astype(np.float64) - b).max() / np.abs(b).max())


GEOMS = [(1, 1, [9, 7], 1), (2, 2, [5, 4, 6, 3], 2), (2, 3, [4, 3, 3, 4, 2], 1), (2, 2, [4, 3, 3, 2], 3),
         (3, 3, [3, 2, 2, 2, 3, 2], 1), (2, 2, [5, 3, 4, 3], 0)]


@pytest.mark.parametrize("geom", GEOMS, ids=lambda g: f"{g[0]}x{g[1]}v-k{g[3]}")
def test_f32_sweeps_are_the_f64_sweeps_to_fp32_rounding(geom):
    """Each output is a sum of 2(k+1) products of fp32-rounded coefficients and fp32 data: against the fp64 result
    on the SAME (float-representable) data the error is at most (2(k+1) + 2) eps32 sum_l (|A|+|B|) max|u|;
    sum_l (|A_jl| + |B_jl|) <= 3 for k <= 3 (Lebesgue-type constant of the GL nodes), so 1.5e-6 max|u| covers it."""
    dx, dv, cells, k = geom
    dom = []
    for a in range(dx + dv):
        dom += [0.0, 1.0 + a] if a < dx else [-2.0 - a, 2.0 + a]
    o = O.Oracle(dx, dv, cells, k, dom)
    f32 = W.random_field(o.shape, seed=W.SEED + k).numpy().astype(np.float32)
    f64 = f32.astype(np.float64)
    for axis in range(dx + (dx if dv >= dx else dv)):
        n = o.D[dx + axis] if axis < dx else o.X
        for kind in ("small", "cfl", "edge"):
            delta = W.delta_table(n, kind, seed=W.SEED + axis, ncells=cells[axis]).numpy()
            got = o.sweep_axis_f32(f32, axis, delta)
            want = o.sweep_axis(f64, axis, delta)
            assert got.dtype == np.float32
            assert rel_inf(got, want) <= 1.5e-6, (axis, kind)
            assert rel_inf(got, want) > 0.0 or k == 0            # it IS single precision arithmetic


@pytest.mark.parametrize("kind", ["int0", "int+1", "int-3", "intwrap", "intmix"])
def test_f32_integer_shifts_are_exact_permutations(kind):
    o = O.Oracle(2, 2, [5, 4, 6, 3], 2, [0, 1, 0, 2, -2, 2, -3, 3])
    f32 = W.random_field(o.shape, seed=5).numpy().astype(np.float32)
    f32.reshape(-1)[::7] = -0.0
    for axis in range(4):
        n = o.D[2 + axis] if axis < 2 else o.X
        delta = W.delta_table(n, kind, seed=W.SEED + axis, ncells=o.cells[axis]).numpy()
        got = o.sweep_axis_f32(f32, axis, delta)
        want = o.sweep_axis(f32.astype(np.float64), axis, delta)      # exact permutation of float-representable data
        assert np.array_equal(got.view(np.int32), want.astype(np.float32).view(np.int32))


def test_f32_density_and_mass_are_fp64_sums_of_the_fp32_values():
    o = O.Oracle(2, 2, [4, 3, 5, 4], 1, [0, 1, 0, 2, -2, 2, -3, 3])
    f32 = W.random_field(o.shape, seed=9).numpy().astype(np.float32)
    assert np.array_equal(o.density_f32(f32), o.density(f32.astype(np.float64)))
    assert o.mass_f32(f32) == o.mass(f32.astype(np.float64))


def test_f32_strang_steps_overlap_with_f64_and_conserve_mass():
    """'the results obtained using single and double precision overlap in the plots'."""
    cfg = W.CONFIGS[0]
    o = O.Oracle(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], threads=O.lib().orc_max_threads())
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)]).numpy()
    f64, f32 = f0.copy(), f0.astype(np.float32)
    m0 = o.mass_f32(f32)
    e64, e32 = [], []
    for _ in range(10):
        f64, _, E64 = o.step(f64, cfg["dt"])
        f32, _, E32 = o.step_f32(f32, cfg["dt"])
        e64.append(o.electric_energy(E64)); e32.append(o.electric_energy(E32))
    assert f32.dtype == np.float32
    assert rel_inf(f32, f64) <= 2e-5
    assert np.abs(np.array(e32) / np.array(e64) - 1).max() <= 1e-3     # the curves of figures 7-8 overlap
    assert abs(o.mass_f32(f32) - m0) <= 2e-6 * abs(m0)


def test_f32_step_is_the_composition_of_its_parts():
    cfg = W.scaled(W.CONFIGS[2], [4, 3, 4, 3, 2])
    o = O.Oracle(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)]).numpy().astype(np.float32)
    dt = cfg["dt"]
    got, rho, E = o.step_f32(f0, dt)
    f = o.advect_x_f32(f0, dt / 2)
    rho2 = o.density_f32(f)
    E2 = o.poisson(rho2)
    f = o.advect_x_f32(o.advect_v_f32(f, E2, dt), dt / 2)
    assert np.array_equal(got, f) and np.array_equal(rho, rho2) and np.array_equal(E, E2)
