"""GPU tests of the double x half step (sweep_fused_cell_kernel<..., DBL>; inside a run of Strang steps the
second x half step of a step is followed directly by the first x half step of the next one, with the same time
increment).  `sldg_steps` runs the two as one pass that applies the sweep pair twice in the order x_1, x_2, x_1, x_2:
same operands and order as two passes, so the result must be BIT-IDENTICAL to the plan without it (and to repeated
`sldg_step` calls), and match the oracle within the 10-step bar.
"""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import oracle as O

pytestmark = pytest.mark.gpu


def rel_inf(g, o):
    return float(np.abs(g.astype(np.float64) - o.astype(np.float64)).max() / np.abs(o).max())


@pytest.fixture(scope="module")
def P():
    import paper_2110_14557_b200 as pkg
    if not torch.cuda.is_available():
        pytest.fail("gpu test without a CUDA device")
    return pkg


def dom_of(dx, dv):
    dom = []
    for a in range(dx + dv):
        dom += [0.0, 1.0 + a] if a < dx else [-2.0 - a, 2.0 + a]
    return dom


# (dim_x, dim_v, cells, degree)
XD_GEOMS = [
    (2, 2, [6, 5, 4, 3], 1),
    (2, 2, [8, 7, 3, 4], 2),          # 7 x_2 cells: ragged groups
    (2, 2, [4, 1, 3, 2], 1),          # a single x_2 cell: every donor is the cell itself
    (2, 2, [4, 2, 2, 3], 2),          # two x_2 cells
    (2, 2, [8, 9, 3, 2], 0),          # degree 0 (D_0 = 8: bulk-copy rule holds)
    (2, 3, [6, 4, 3, 2, 2], 1),       # 2x3v
    (2, 2, [64, 5, 2, 2], 2),         # D_0 = 192 as in BASELINE cfg2
    (2, 2, [6, 5, 4, 3], 3),          # degree 3: no double pass (registers) -> plain plan
    (2, 2, [5, 4, 3, 2], 0),          # D_0 = 5: rows not a multiple of 16 B -> plain plan
]


@pytest.mark.parametrize("geom", XD_GEOMS, ids=lambda g: f"{g[0]}x{g[1]}v-{'x'.join(map(str, g[2]))}-k{g[3]}")
@pytest.mark.parametrize("dt", [0.05, 0.9])                     # |x shift| < 1 cell / up to ~10 cells (wraps)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_steps_with_double_x_pass_are_bitwise_the_plain_plan(P, geom, dt, prec):
    dx, dv, cells, k = geom
    dom = dom_of(dx, dv)
    o = O.Oracle(dx, dv, cells, k, dom, threads=O.lib().orc_max_threads())
    f0 = W.random_field(o.shape, seed=41 + k)
    if prec == "f32":
        f0 = f0.to(torch.float32)
    outs = []
    # (x_double, fuse_v, cell_rows, cell_threads, nsteps)
    for xd, fv, rows, thr, n in ((0, 0, 0, 64, 4), (1, 0, 0, 64, 4), (1, 2, 1, 128, 4), (1, 2, 3, 32, 4), (1, 0, 2, 64, 4)):
        g = P.Sldg(dx, dv, cells, k, dom, precision=prec)
        g.set_option("graph", 0); g.set_option("x_double", xd); g.set_option("fuse_v", fv)
        g.set_option("cell_rows", rows); g.set_option("cell_threads", thr)
        fg = f0.to(g.device).contiguous()
        n0 = g.launch_count()
        g.steps(fg, dt, n)
        outs.append((fg.cpu().numpy(), g.launch_count() - n0))
    for x, _ in outs[1:]:
        assert np.array_equal(outs[0][0], x)
    doubled = k <= 2 and (cells[0] * (k + 1) * (k + 1) * (8 if prec == "f64" else 4)) % 16 == 0
    if doubled:
        assert outs[1][1] < outs[0][1]                              # the merged passes really ran
    else:
        assert outs[1][1] == outs[0][1]
    if prec == "f64":
        want = f0.numpy()
        for _ in range(4):
            want, _, _ = o.step(want, dt)
        assert rel_inf(outs[0][0], want) <= 1e-10


# dim_x = 3: the double x_1x_2x_3 pass (sldg_sweep_fused3d.cu)
X3D_GEOMS = [
    ([4, 5, 3, 2, 2, 2], 1),          # 5 x_2 cells: strips of 1..5 cells, ragged last strip
    ([20, 7, 3, 2, 2, 2], 1),         # D_0 = 40 as in BASELINE cfg4; 7 x_2 cells
    ([6, 5, 1, 2, 3, 2], 1),          # a single x_3 cell: the wrap cells are the only donor pairs
    ([6, 5, 2, 2, 3, 2], 1),          # two x_3 cells
    ([4, 1, 3, 2, 2, 3], 1),          # a single x_2 cell: every halo cell is the cell itself
    ([4, 2, 3, 2, 2, 3], 1),          # two x_2 cells: the input range wraps around the axis
    ([8, 6, 4, 2, 3, 2], 0),          # degree 0 (D_0 = 8: bulk-copy rule holds)
    ([5, 4, 3, 2, 2, 2], 0),          # degree 0, D_0 = 5: rows not a multiple of 16 B -> plain plan
    ([3, 2, 2, 3, 2, 2], 2),          # degree 2: no fused x_1x_2x_3 passes at all -> plain plan
]


@pytest.mark.parametrize("geom", X3D_GEOMS, ids=lambda g: f"{'x'.join(map(str, g[0]))}-k{g[1]}")
@pytest.mark.parametrize("dt", [0.03, 0.9])                     # |x shift| < 1 cell / up to ~10 cells (wraps)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_steps_with_double_x3_pass_are_bitwise_the_plain_plan(P, geom, dt, prec):
    cells, k = geom
    dom = dom_of(3, 3)
    o = O.Oracle(3, 3, cells, k, dom, threads=O.lib().orc_max_threads())
    f0 = W.random_field(o.shape, seed=43 + k)
    if prec == "f32":
        f0 = f0.to(torch.float32)
    outs = []
    # (x_double, fuse_v3, f3d_threads, f3_stages, nsteps)
    # x_double = 2: the dim_x = 3 double pass is planned only when forced (measured slower than two passes on B200)
    for xd, fv3, thr, st, n in ((0, 0, 128, 3, 4), (2, 0, 128, 3, 4), (2, 2, 2 * cells[0], 2, 4), (2, 2, 3 * cells[0], 4, 4),
                                (2, 0, 256, 3, 4), (2, 2, 128, 3, 3), (1, 2, 128, 3, 3)):
        g = P.Sldg(3, 3, cells, k, dom, precision=prec)
        g.set_option("graph", 0); g.set_option("x_double", xd); g.set_option("fuse_v3", fv3)
        g.set_option("f3d_threads", min(256, thr)); g.set_option("f3_stages", st)
        fg = f0.to(g.device).contiguous()
        n0 = g.launch_count()
        g.steps(fg, dt, n)
        outs.append((fg.cpu().numpy(), g.launch_count() - n0, n))
    for x, _, n in outs[1:5]:
        assert np.array_equal(outs[0][0], x)
    assert np.array_equal(outs[5][0], outs[6][0])                   # three steps, one-pass v advection on both sides
    doubled = k <= 1 and (cells[0] * (k + 1) * (k + 1) * (8 if prec == "f64" else 4)) % 16 == 0
    if doubled:
        assert outs[1][1] < outs[0][1] and outs[5][1] < outs[6][1]  # the merged passes really ran
    else:
        assert outs[1][1] == outs[0][1]
    if prec == "f64":
        want = f0.numpy()
        for _ in range(4):
            want, _, _ = o.step(want, dt)
        assert rel_inf(outs[0][0], want) <= 1e-10


@pytest.mark.parametrize("n", [2, 3, 5])
def test_steps_equal_repeated_single_steps_with_the_double_x3_pass(P, n):
    cfg = W.scaled(W.CONFIGS[3], [6, 5, 4, 6, 4, 4])
    o = O.Oracle(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], threads=1)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
    g.set_option("graph", 0); g.set_option("fuse_v3", 2); g.set_option("x_double", 2)
    fa, fb = f0.to(g.device).contiguous(), f0.to(g.device).contiguous()
    for _ in range(n):
        g.step(fa, cfg["dt"])
    g.timing_enable(True); g.timing_read()
    g.steps(fb, cfg["dt"], n)
    kinds, _ = g.timing_read()
    assert torch.equal(fa, fb)
    assert kinds["sweep_fused_x3_double"][0] == n - 1


@pytest.mark.parametrize("n", [2, 3, 5])
def test_steps_equal_repeated_single_steps_with_the_double_pass(P, n):
    cfg = W.scaled(W.CONFIGS[1], [12, 10, 8, 8])
    o = O.Oracle(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], threads=1)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
    g.set_option("graph", 0)
    fa, fb = f0.to(g.device).contiguous(), f0.to(g.device).contiguous()
    for _ in range(n):
        g.step(fa, cfg["dt"])
    g.steps(fb, cfg["dt"], n)
    assert torch.equal(fa, fb)


@pytest.mark.parametrize("geom", [(2, 2, [12, 10, 8, 8], 2), (2, 3, [8, 8, 6, 6, 4], 1), (3, 3, [6, 4, 4, 6, 4, 4], 1)],
                         ids=lambda g: f"{g[0]}x{g[1]}v-k{g[3]}")
@pytest.mark.parametrize("n", [0, 2, 5])
@pytest.mark.parametrize("fuse_v,x_double", [(0, 0), (2, 0), (2, 1), (0, 1), (2, 2)])
def test_plan_query_counts_are_those_of_the_real_calls(P, geom, n, fuse_v, x_double):
    """The host-only sldg_plan_query (tests/test_plan.py checks its budgets on the CPU) must report exactly the sweep
    launches the real sldg_step / sldg_steps make: per-kind launch counts from the library's event instrumentation."""
    dx, dv, cells, k = geom
    dom = dom_of(dx, dv)
    g = P.Sldg(dx, dv, cells, k, dom)
    g.set_option("graph", 0); g.set_option("fuse_v", fuse_v); g.set_option("x_double", x_double)
    f = W.random_field(g.shape, seed=2).to(g.device).contiguous()
    dt = 0.01                                                      # every x shift below one cell
    g.timing_enable(True); g.timing_read()
    if n == 0:
        g.step(f, dt)
    else:
        g.steps(f, dt, n)
    kinds, _ = g.timing_read()
    g.timing_enable(False)
    want = P.plan_query(dx, dv, cells, k, n, shifts_below_one=True, fuse_v=fuse_v, x_double=x_double)
    sweeps = sum(v[0] for name, v in kinds.items() if name.startswith("sweep"))
    assert sweeps == want["x_passes"] + want["v_passes"]
    assert kinds["sweep_fused_v"][0] + kinds["sweep_slow_axis"][0] >= want["v_passes"]
    assert kinds["table_uploads"][0] == dx                         # the x shift-table uploads (one event per axis)
    assert kinds["copies"][0] == want["copies"] == 0               # and no whole-array copy of f
    assert kinds["rho"][0] == max(1, n)


@pytest.mark.parametrize("ci", [1, 2, 3], ids=lambda i: W.CONFIGS[i]["name"])
def test_merged_steps_equal_single_steps_at_full_size(P, ci):
    """BASELINE configs 2-4 at FULL size in the launch configuration bench.py times (sldg_steps: double x half steps,
    fused v passes, alternating buffers): three merged steps, repeated, must give the bits of three sldg_step calls.
    Long walks under memory contention are where a missing proxy fence once showed."""
    cfg = W.CONFIGS[ci]
    g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
    f0 = g.empty_field()
    W.initial_data(cfg, [g.node_coords(a) for a in range(g.d)], device=f0.device, out=f0)
    W.perturb_inplace(f0)
    ref = f0.clone()
    for _ in range(3):
        g.step(ref, cfg["dt"])
    m_ref = g.mass(ref)
    for rep in range(3):
        f = f0.clone()
        g.steps(f, cfg["dt"], 3)
        assert torch.equal(f, ref), (rep, int((f != ref).sum()))
        del f
    assert abs(m_ref - g.mass(f0)) <= 1e-12 * abs(m_ref)


def _bits_checksum(f):
    """Order-independent 2 x 64-bit checksum of the bit patterns of a device array, slab by slab (no |f|-sized
    temporary): wrapping sums of the words and of the words mixed with their slab index."""
    import torch
    h1 = torch.zeros((), dtype=torch.int64, device=f.device)
    h2 = torch.zeros((), dtype=torch.int64, device=f.device)
    flat = f.view(f.shape[0], -1)
    for i in range(flat.shape[0]):
        w = flat[i].view(torch.int64)
        s = w.sum()
        h1 += s
        h2 += (w ^ (w >> 17)).sum() * (2 * i + 1)
    return int(h1.item()), int(h2.item())


def test_merged_steps_equal_single_steps_at_the_hbm_filling_size(P):
    """BASELINE config 5 (56.6 GB + as much workspace): a third full-size buffer does not fit, so three sldg_step calls and
    sldg_steps(3) (alternating buffers, the one-pass v advection, the closing half step that restores the parity) start
    from the same regenerated data and are compared through a checksum of all bit patterns."""
    cfg = W.CONFIGS[4]
    g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
    coords = [g.node_coords(a) for a in range(g.d)]
    f = g.empty_field()
    sums = []
    for multi in (0, 1, 1):
        W.initial_data(cfg, coords, device=f.device, out=f)
        W.perturb_inplace(f)
        if multi:
            g.steps(f, cfg["dt"], 3)
        else:
            for _ in range(3):
                g.step(f, cfg["dt"])
        sums.append(_bits_checksum(f))
    assert sums[0] == sums[1] == sums[2], sums
