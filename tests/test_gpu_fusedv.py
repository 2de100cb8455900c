"""GPU tests of the fused v_1+v_2 pass (sldg_sweep_fusedv.cu; P:88-92 -- E does not change
during the v sweeps, so the two sweeps can share one pass over f).

The fused pass does, per value, the arithmetic of the slow-axis walk on v_1 and then on v_2 (same operands, same
order), so (i) fused and unfused plans must agree BIT FOR BIT, for every tiling of the fused kernel, and (ii) both
must match the oracle within the per-sweep bar.  Integer shifts stay exact permutations.
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


def make_pair(P, dx, dv, cells, k, precision="f64"):
    dom = []
    for a in range(dx + dv):
        dom += [0.0, 1.0 + a] if a < dx else [-2.0 - a, 2.0 + a]
    return (P.Sldg(dx, dv, cells, k, dom, precision=precision),
            O.Oracle(dx, dv, cells, k, dom, threads=O.lib().orc_max_threads()))


# (dim_x, dim_v, cells, degree)
FV_GEOMS = [
    (2, 2, [4, 4, 6, 5], 1),          # X = 64: whole tiles
    (2, 2, [5, 3, 7, 4], 1),          # X = 60: ragged last tile (TMA zero fill)
    (2, 2, [6, 4, 5, 3], 2),          # k = 2: first block streamed in again
    (2, 2, [3, 2, 1, 4], 2),          # a single v_1 cell: both donors are the cell itself
    (2, 2, [4, 2, 5, 1], 1),          # a single v_2 cell
    (2, 2, [6, 5, 4, 3], 0),          # degree 0
    (2, 3, [6, 4, 5, 4, 3], 1),       # 2x3v: v_3 idle, 6 planes
    (3, 3, [4, 3, 5, 3, 4, 2], 1),    # 3x3v: fused v_1+v_2, then v_3 by the walk
    (2, 2, [3, 3, 4, 3], 2),          # X = 81 (odd): rows not a multiple of 16 B -> planner falls back
    (2, 2, [6, 4, 5, 3], 3),          # degree 3: 256-thread blocks, A_2, B_2 in shared memory, first block streamed in again
    (2, 2, [6, 4, 5, 3], 4),          # degree 4: not fused (registers) -> planner falls back
    (2, 3, [8, 4, 16, 3, 2], 3),      # degree 3, N_1 = 16 as in the bump-on-tail workload (bot_5d_k3_16)
    (2, 2, [16, 12, 20, 6], 1),       # D_1 = 40 as in BASELINE cfg4, 24 tiles
    (2, 2, [8, 4, 64, 3], 2),         # N_1 = 64, k = 2 as in BASELINE cfg2: 512 threads, 8 x nodes per tile
]


def run_plans(g, f0, E, dt, plans):
    outs = []
    for fuse, wx, stages, ppb, l2, cps in plans:
        g.set_option("fuse_v", fuse); g.set_option("fv_wx", wx); g.set_option("fv_stages", stages)
        g.set_option("fv_ppb", ppb); g.set_option("fv_l2", l2); g.set_option("fv_cps", cps)
        fg = f0.to(g.device).contiguous()
        n0 = g.launch_count()
        g.advect_v(fg, E, dt)
        outs.append((fg.cpu().numpy(), g.launch_count() - n0))
    return outs


# (fuse_v: 0 never, 1 auto, 2 whenever the shape allows; fv_wx, fv_stages, fv_ppb, fv_l2, fv_cps: v_2 cells per copy)
PLANS = ((0, 0, 0, 0, 2, 1), (2, 0, 0, 0, 2, 1), (2, 2, 3, 1, 0, 2), (2, 4, 5, 2, 1, 3), (2, 8, 2, 3, 3, 1), (2, 16, 9, 0, 2, 4),
         (2, 0, 4, 0, 2, 2), (1, 0, 0, 0, 2, 1))


@pytest.mark.parametrize("geom", FV_GEOMS, ids=lambda g: f"{g[0]}x{g[1]}v-{'x'.join(map(str, g[2]))}-k{g[3]}")
@pytest.mark.parametrize("amp", [0.02, 3.0, 40.0])
def test_fused_v_pass_agrees_bitwise_with_separate_sweeps_and_matches_oracle(P, geom, amp):
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k)
    f0 = W.random_field(o.shape, seed=17 + k)
    dt = 0.1
    hv = (2 * (2.0 + dx)) / cells[dx]
    E = W.random_E(dx, o.xshape, seed=5, amplitude=amp * hv / dt)      # |delta| up to amp cells, both signs
    outs = run_plans(g, f0, E.to(g.device), dt, PLANS)
    for x, _ in outs[1:]:
        assert np.array_equal(outs[0][0], x)
    assert rel_inf(outs[0][0], o.advect_v(f0.numpy(), E.numpy(), dt)) <= TOL_SWEEP * dx
    fusable = k <= 3 and (o.xshape and int(np.prod(o.xshape)) % 2 == 0)
    if fusable:
        assert outs[1][1] < outs[0][1]                                  # the fused pass really ran (one launch fewer)
    else:
        assert outs[1][1] == outs[0][1]
    assert outs[-1][1] == outs[0][1]                                    # auto rule: too few walks on these small grids


def test_fused_v_integer_shifts_are_exact(P):
    """E = m h_v / dt with dyadic h_v, dt: delta = -m exactly; -0.0 and NaN payloads survive."""
    dom = [0, 1.0, 0, 1.0, -3.0, 3.0, -1.5, 1.5]
    outs = []
    for fuse in (2, 0):
        g = P.Sldg(2, 2, [4, 6, 8, 4], 1, dom)                          # h_v = 0.75
        o = O.Oracle(2, 2, [4, 6, 8, 4], 1, dom, threads=1)
        g.set_option("fuse_v", fuse)
        f0 = W.random_field(o.shape, seed=11)
        f0.view(-1)[::7] = -0.0
        f0.view(-1)[3::1001] = float("nan")
        dt = 0.25
        E = np.empty((2,) + o.xshape)
        E[0] = 2 * 0.75 / dt
        E[1] = -1 * 0.75 / dt
        fg = f0.to(g.device).contiguous()
        g.advect_v(fg, torch.from_numpy(E).to(g.device), dt)
        want = np.roll(np.roll(f0.numpy(), -2 * 2, axis=1), 1 * 2, axis=0)
        assert np.array_equal(fg.cpu().numpy().view(np.int64), want.view(np.int64))
        outs.append(fg.cpu().numpy())


@pytest.mark.parametrize("geom", [(2, 2, [6, 4, 5, 3], 2), (2, 3, [6, 4, 5, 4, 3], 1), (3, 3, [4, 3, 5, 3, 4, 2], 1),
                                  (2, 2, [8, 4, 6, 5], 1)],
                         ids=lambda g: f"{g[0]}x{g[1]}v-k{g[3]}")
def test_fused_v_single_precision_agrees_bitwise_and_matches_fp32_oracle(P, geom):
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k, precision="f32")
    f0 = W.random_field(o.shape, seed=23).to(torch.float32)
    dt = 0.1
    hv = (2 * (2.0 + dx)) / cells[dx]
    E = W.random_E(dx, o.xshape, seed=6, amplitude=2.5 * hv / dt)
    outs = run_plans(g, f0, E.to(g.device), dt, ((0, 0, 0, 0, 2, 1), (2, 0, 0, 0, 2, 1), (2, 4, 3, 1, 0, 2), (2, 8, 6, 2, 2, 3), (2, 0, 5, 0, 2, 2)))
    for x, _ in outs[1:]:
        assert np.array_equal(outs[0][0], x)
    assert outs[1][1] < outs[0][1]
    assert rel_inf(outs[0][0], o.advect_v_f32(f0.numpy(), E.numpy(), dt)) <= 2e-6 * dx


def small_cfgs():
    c = W.CONFIGS
    return [c[0], W.scaled(c[1], [12, 10, 8, 8]), W.scaled(c[2], [8, 8, 6, 6, 4]), W.scaled(c[3], [6, 4, 4, 6, 4, 4])]


@pytest.mark.parametrize("cfg", small_cfgs(), ids=lambda c: c["name"])
@pytest.mark.parametrize("n", [1, 3, 4])
def test_steps_with_and_without_fused_v_agree_bitwise(P, cfg, n):
    """Whole Strang steps (sldg_step and the multi-step sldg_steps, whose buffer-flip parities change with the number
    of v passes) give the same bits with the fused v pass on and off, and end in the caller's buffer."""
    o = O.Oracle(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], threads=1)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    outs = []
    for fuse, multi in ((0, 0), (2, 0), (2, 1), (0, 1)):
        g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
        g.set_option("graph", 0); g.set_option("fuse_v", fuse)
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
    # dim_x = 2: a single step must end in the caller's buffer, so the pass saved in v is spent in x (equal counts);
    # consecutive steps through sldg_steps alternate buffers and keep the saving.  dim_x = 3: always fewer.
    assert outs[1][1] <= outs[0][1] and outs[2][1] <= outs[3][1]
    if n >= 3 or cfg["dim_x"] == 3:
        assert outs[2][1] < outs[3][1]


@pytest.mark.parametrize("geom", [(2, 2, [5, 3, 7, 4], 1), (2, 2, [6, 4, 5, 3], 2), (3, 3, [4, 3, 5, 3, 4, 2], 1)],
                         ids=lambda g: f"{g[0]}x{g[1]}v-k{g[3]}")
def test_fused_v_pass_stays_inside_the_field(P, geom):
    """Canary bands around the caller's f (compute-sanitizer is not available on the GPU pool): the fused pass, whose
    ragged last x tile is zero-filled by the tensor copy and whose stores are predicated per thread, must not touch a
    byte outside f; an out-of-range store into the workspace copy would break the bitwise plan equivalence above."""
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k)
    g.set_option("fuse_v", 2); g.set_option("graph", 0)
    n = int(np.prod(o.shape))
    guard = 4096
    big = torch.full((n + 2 * guard,), float("nan"), dtype=torch.float64, device=g.device)
    f = big[guard:guard + n].view(o.shape)
    f0 = W.random_field(o.shape, seed=3)
    f.copy_(f0)
    E = W.random_E(dx, o.xshape, seed=9, amplitude=25.0).to(g.device)
    g.advect_v(f, E, 0.1)
    g.steps(f, 0.05, 3)
    assert bool(torch.isnan(big[:guard]).all()) and bool(torch.isnan(big[guard + n:]).all())
    assert bool(torch.isfinite(f).all())
    want = o.advect_v(f0.numpy(), E.cpu().numpy(), 0.1)
    for _ in range(3):
        want, _, _ = o.step(want, 0.05)
    assert rel_inf(f.cpu().numpy(), want) <= 1e-10


def test_fused_v_pass_inside_a_captured_step_graph(P):
    """The tensor map of the fused pass is a by-value kernel parameter built on the host at launch time: a Strang step
    captured into a CUDA graph (option graph = 2) and replayed must give the bits of plain launches."""
    cfg = W.scaled(W.CONFIGS[1], [12, 10, 8, 8])
    o = O.Oracle(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], threads=1)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    outs = []
    for graph in (0, 2):
        g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
        g.set_option("fuse_v", 2); g.set_option("graph", graph)
        fg = f0.to(g.device).contiguous()
        for _ in range(4):
            g.step(fg, cfg["dt"])
        outs.append(fg.cpu().numpy())
    assert np.array_equal(outs[0], outs[1])


def test_fused_v_ring_under_drift_long_multi_plane_walks(P):
    """Regression for a cross-proxy write-after-read race: a ring slot read by the generic proxy was handed back to the
    TMA (async proxy) without a proxy fence, so single lanes could read rows of the NEXT copy.  It needed warps that
    drift apart (long walks over many planes, few ring slots, memory contention) and showed only at full size, as a
    mass error of 1e-9 in tests/test_gpu_fullsize.py.  Here: 1.1 GB, 144 blocks walking 64 planes each, strong seeded
    field, several ring depths; every run must give the bits of the separate walks."""
    dx, dv, cells, k = 2, 3, [24, 24, 20, 12, 32], 1
    g, o = make_pair(P, dx, dv, cells, k)
    f0 = W.random_field(g.shape, seed=77, device=g.device)
    hv = (2 * (2.0 + dx)) / cells[dx]
    E = W.random_E(dx, g.xshape, seed=12, amplitude=3.0 * hv / 0.1, device=g.device)
    g.set_option("fuse_v", 0)
    want = f0.clone()
    g.advect_v(want, E, 0.1)
    g.set_option("fuse_v", 2)
    for stages, ppb in ((3, 64), (4, 64), (8, 64), (3, 16), (0, 0)):
        g.set_option("fv_stages", stages); g.set_option("fv_ppb", ppb)
        for _ in range(4):
            got = f0.clone()
            g.advect_v(got, E, 0.1)
            assert torch.equal(got, want), (stages, ppb, int((got != want).sum()))
