"""GPU tests of the fused v_1+v_2+v_3 pass (sldg_sweep_fusedv3.cu; SURVEY 8(a) rows a5/a6 for the 3x3v case the paper
focuses on: E does not change during the v sweeps, so all three can share one pass over f).

The fused pass does, per value, the arithmetic of the slow-axis walk on v_1, v_2 and v_3 in turn (same operands, same
order), so (i) fused and unfused plans must agree BIT FOR BIT, for every tiling (x nodes per tile, strip size, ring
depth), and (ii) both must match the oracle within the per-sweep bar.  Integer shifts stay exact permutations.
"""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import oracle as O

pytestmark = pytest.mark.gpu

TOL_SWEEP = 1e-12


def rel_inf(g, o):
    return float(np.abs(g.astype(np.float64) - o.astype(np.float64)).max() / np.abs(o).max())


@pytest.fixture(scope="module")
def P():
    import paper_2110_14557_b200 as pkg
    if not torch.cuda.is_available():
        pytest.fail("gpu test without a CUDA device")
    return pkg


def make_pair(P, cells, k, precision="f64"):
    dom = []
    for a in range(6):
        dom += [0.0, 1.0 + a] if a < 3 else [-2.0 - a, 2.0 + a]
    return (P.Sldg(3, 3, cells, k, dom, precision=precision),
            O.Oracle(3, 3, cells, k, dom, threads=O.lib().orc_max_threads()))


# (cells, degree)
FV3_GEOMS = [
    ([4, 2, 2, 5, 6, 4], 1),          # X = 64: whole tiles; 6 v_2 cells: strips of 1..5 pairs, ragged last strip
    ([5, 3, 1, 3, 7, 3], 1),          # X = 60: ragged last x tile (TMA zero fill); 7 v_2 cells
    ([2, 2, 2, 1, 4, 3], 1),          # a single v_1 cell: both donors are the cell itself
    ([2, 2, 2, 4, 1, 3], 1),          # a single v_2 cell: the pair is (cell, cell)
    ([2, 2, 2, 4, 3, 1], 1),          # a single v_3 cell
    ([4, 2, 2, 5, 6, 4], 0),          # degree 0
    ([3, 3, 1, 3, 4, 2], 0),          # degree 0, X = 9 (odd): rows not a multiple of 16 B -> planner falls back
    ([2, 2, 2, 20, 5, 3], 1),         # D_1 = 40 as in BASELINE cfg4 / cfg5: 320 threads at 16 x nodes per tile
    ([3, 2, 2, 4, 3, 3], 2),          # degree 2: not fused (registers) -> planner falls back
]

# (fuse_v3: 0 never / 2 whenever the shape allows, fv3_wx, fv3_strip, fv3_slots[, fv3_pw: dedicated producer warp]); plan 0 = three
# separate walks; the last plan is the automatic rule
PLANS = ((0, 0, 0, 0), (2, 0, 0, 0), (2, 2, 1, 3), (2, 4, 2, 2), (2, 8, 3, 5), (2, 16, 5, 0), (2, 0, 4, 4),
         (2, 0, 0, 0, 1), (2, 8, 2, 2, 1), (2, 16, 5, 3, 1), (2, 4, 1, 5, 1), (1, 0, 0, 0))


def run_plans(g, f0, E, dt, plans):
    outs = []
    for fuse3, wx, strip, slots, *rest in plans:
        g.set_option("fuse_v", 0); g.set_option("fuse_v3", fuse3); g.set_option("fv3_wx", wx)
        g.set_option("fv3_strip", strip); g.set_option("fv3_slots", slots); g.set_option("fv3_pw", rest[0] if rest else 0)
        fg = f0.to(g.device).contiguous()
        n0 = g.launch_count()
        g.advect_v(fg, E, dt)
        outs.append((fg.cpu().numpy(), g.launch_count() - n0))
    return outs


@pytest.mark.parametrize("geom", FV3_GEOMS, ids=lambda g: f"{'x'.join(map(str, g[0]))}-k{g[1]}")
@pytest.mark.parametrize("amp", [0.02, 3.0, 40.0])
def test_fused_v3_pass_agrees_bitwise_with_separate_sweeps_and_matches_oracle(P, geom, amp):
    cells, k = geom
    g, o = make_pair(P, cells, k)
    f0 = W.random_field(o.shape, seed=19 + k)
    dt = 0.1
    hv = (2 * (2.0 + 3)) / cells[3]
    E = W.random_E(3, o.xshape, seed=5, amplitude=amp * hv / dt)       # |delta| up to amp cells, both signs
    outs = run_plans(g, f0, E.to(g.device), dt, PLANS)
    for x, _ in outs[1:]:
        assert np.array_equal(outs[0][0], x)
    assert rel_inf(outs[0][0], o.advect_v(f0.numpy(), E.numpy(), dt)) <= TOL_SWEEP * 3
    fusable = k <= 1 and int(np.prod(o.xshape)) % 2 == 0
    if fusable:
        assert outs[1][1] < outs[0][1]                                  # the fused pass really ran (two launches fewer)
    else:
        assert outs[1][1] == outs[0][1]
    assert outs[-1][1] == outs[0][1]                                    # auto rule: too few walks on these small grids


def test_fused_v3_integer_shifts_are_exact(P):
    """E = m h_v / dt with dyadic h_v, dt: delta = -m exactly on all three axes; -0.0 and NaN payloads survive."""
    dom = [0, 1.0, 0, 1.0, 0, 1.0, -3.0, 3.0, -1.5, 1.5, -0.75, 0.75]
    cells = [2, 4, 2, 8, 4, 2]                                          # h_v = 0.75 on every v axis
    g = P.Sldg(3, 3, cells, 1, dom)
    o = O.Oracle(3, 3, cells, 1, dom, threads=1)
    g.set_option("fuse_v3", 2)
    f0 = W.random_field(o.shape, seed=11)
    f0.view(-1)[::7] = -0.0
    f0.view(-1)[3::1001] = float("nan")
    dt = 0.25
    E = np.empty((3,) + o.xshape)
    E[0] = 2 * 0.75 / dt
    E[1] = -1 * 0.75 / dt
    E[2] = 3 * 0.75 / dt
    fg = f0.to(g.device).contiguous()
    n0 = g.launch_count()
    g.advect_v(fg, torch.from_numpy(E).to(g.device), dt)
    assert g.launch_count() - n0 == 4                                   # three table kernels + ONE pass
    want = np.roll(np.roll(np.roll(f0.numpy(), -2 * 2, axis=2), 1 * 2, axis=1), -3 * 2, axis=0)
    assert np.array_equal(fg.cpu().numpy().view(np.int64), want.view(np.int64))


@pytest.mark.parametrize("geom", [([4, 2, 2, 5, 6, 4], 1), ([5, 3, 1, 3, 7, 3], 1), ([4, 2, 2, 5, 6, 4], 0)],
                         ids=lambda g: f"{'x'.join(map(str, g[0]))}-k{g[1]}")
def test_fused_v3_single_precision_agrees_bitwise_and_matches_fp32_oracle(P, geom):
    cells, k = geom
    g, o = make_pair(P, cells, k, precision="f32")
    f0 = W.random_field(o.shape, seed=23).to(torch.float32)
    dt = 0.1
    hv = (2 * (2.0 + 3)) / cells[3]
    E = W.random_E(3, o.xshape, seed=6, amplitude=2.5 * hv / dt)
    outs = run_plans(g, f0, E.to(g.device), dt, ((0, 0, 0, 0), (2, 0, 0, 0), (2, 4, 1, 3), (2, 8, 3, 2), (2, 0, 5, 6)))
    for x, _ in outs[1:]:
        assert np.array_equal(outs[0][0], x)
    if int(np.prod(o.xshape)) % 4 == 0:
        assert outs[1][1] < outs[0][1]
    assert rel_inf(outs[0][0], o.advect_v_f32(f0.numpy(), E.numpy(), dt)) <= 2e-6 * 3


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_steps_with_and_without_fused_v3_agree_bitwise(P, n):
    """Whole Strang steps (sldg_step and sldg_steps, whose buffer-flip parities change with the number of v passes) give
    the same bits with the one-pass v advection forced on and off, end in the caller's buffer, and match the oracle."""
    cfg = W.scaled(W.CONFIGS[3], [6, 4, 4, 6, 4, 4])
    o = O.Oracle(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], threads=O.lib().orc_max_threads())
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    outs = []
    for fuse3, multi in ((0, 0), (2, 0), (2, 1), (0, 1)):
        g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
        g.set_option("graph", 0); g.set_option("fuse_v3", fuse3)
        fg = f0.to(g.device).contiguous()
        n0 = g.launch_count()
        if multi:
            g.steps(fg, cfg["dt"], n)
        else:
            for _ in range(n):
                g.step(fg, cfg["dt"])
        outs.append((fg.cpu().numpy(), g.launch_count() - n0))
    for x, _ in outs[1:]:
        assert np.array_equal(outs[0][0], x)
    if n >= 2:
        assert outs[2][1] < outs[3][1]                                  # sldg_steps keeps the saving
    want = f0.numpy()
    for _ in range(n):
        want, _, _ = o.step(want, cfg["dt"])
    assert rel_inf(outs[0][0], want) <= 1e-10


def test_fused_v3_pass_stays_inside_the_field(P):
    """Canary bands around the caller's f: the ragged last x tile is zero-filled by the tensor copy and the stores are
    predicated per thread; no byte outside f may change."""
    cells, k = [5, 3, 1, 3, 7, 3], 1
    g, o = make_pair(P, cells, k)
    g.set_option("fuse_v3", 2); g.set_option("graph", 0)
    n = int(np.prod(o.shape))
    guard = 4096
    big = torch.full((n + 2 * guard,), float("nan"), dtype=torch.float64, device=g.device)
    f = big[guard:guard + n].view(o.shape)
    f0 = W.random_field(o.shape, seed=3)
    f.copy_(f0)
    E = W.random_E(3, o.xshape, seed=9, amplitude=25.0).to(g.device)
    g.advect_v(f, E, 0.1)
    g.steps(f, 0.05, 3)
    assert bool(torch.isnan(big[:guard]).all()) and bool(torch.isnan(big[guard + n:]).all())
    assert bool(torch.isfinite(f).all())
    want = o.advect_v(f0.numpy(), E.cpu().numpy(), 0.1)
    for _ in range(3):
        want, _, _ = o.step(want, 0.05)
    assert rel_inf(f.cpu().numpy(), want) <= 1e-10


def test_fused_v3_ring_under_drift_long_walks(P):
    """The ring-slot hand-over (generic-proxy reads, async-proxy refill; see the regression of sldg_sweep_fusedv.cu) under
    long walks with few slots: 0.9 GB, 40 v_3 cells, strong seeded field, several ring depths and strip sizes; every run
    must give the bits of the separate walks."""
    cells, k = [8, 8, 6, 20, 10, 40], 1
    g, o = make_pair(P, cells, k)
    f0 = W.random_field(g.shape, seed=77, device=g.device)
    hv = (2 * (2.0 + 3)) / cells[3]
    E = W.random_E(3, g.xshape, seed=12, amplitude=3.0 * hv / 0.1, device=g.device)
    g.set_option("fuse_v", 0); g.set_option("fuse_v3", 0)
    want = f0.clone()
    g.advect_v(want, E, 0.1)
    g.set_option("fuse_v3", 2)
    for slots, strip, pw in ((2, 1, 0), (3, 5, 0), (4, 2, 0), (0, 0, 0), (2, 1, 1), (3, 5, 1), (0, 0, 1)):
        g.set_option("fv3_slots", slots); g.set_option("fv3_strip", strip); g.set_option("fv3_pw", pw)
        for _ in range(3):
            got = f0.clone()
            g.advect_v(got, E, 0.1)
            assert torch.equal(got, want), (slots, strip, pw, int((got != want).sum()))
