"""GPU parity: the CUDA path (through the C-ABI, via the ctypes binding) against the CPU oracle, element by
element on the same seeded inputs.  Bars (BASELINE.json north_star): max|g-o|/max|o| <= 1e-12 per sweep,
<= 1e-10 after 10 Strang steps, bit-exact for integer shifts.
"""
import math

import numpy as np
import pytest
import torch

import workloads as W
from oracle import oracle as O

pytestmark = pytest.mark.gpu

TOL_SWEEP = 1e-12
TOL_STEPS = 1e-10


def rel_inf(g, o):
    return float(np.abs(g - o).max() / np.abs(o).max())


@pytest.fixture(scope="module")
def P():
    import paper_2110_14557_b200 as pkg
    if not torch.cuda.is_available():
        pytest.fail("gpu test without a CUDA device")
    return pkg


def make_pair(P, dx, dv, cells, k, dom=None):
    if dom is None:
        dom = []
        for a in range(dx + dv):
            dom += [0.0, 1.0 + a] if a < dx else [-2.0 - a, 2.0 + a]
    return P.Sldg(dx, dv, cells, k, dom), O.Oracle(dx, dv, cells, k, dom, threads=O.lib().orc_max_threads())


def pair_of_cfg(P, cfg):
    return make_pair(P, cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])


# --------------------------------------------------------------- constants

@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_AB_and_nodes_match_oracle(P, k):
    g, o = make_pair(P, 1, 1, [3, 2], k)
    for a in range(2):
        assert np.abs(g.node_coords(a) - o.node_coords(a)).max() <= 4e-16 * 5
    for alpha in [0.0, 1e-12, 1e-3, 0.123, 0.3, 0.5, 0.77, 0.999, 1 - 1e-12]:
        A, B = g.AB(alpha)
        Ao, Bo = O.AB(k, alpha)
        assert np.abs(A - Ao).max() < 5e-14 and np.abs(B - Bo).max() < 5e-14, (k, alpha)


# --------------------------------------------------------------- single sweeps through the test hook

GEOMS = [
    # dx, dv, cells, k      (several tiles, ragged tails, odd sizes, all degrees)
    (1, 1, [37, 23], 1),
    (1, 2, [16, 5, 7], 2),
    (2, 2, [8, 8, 16, 16], 1),        # BASELINE config 1
    (2, 2, [7, 5, 6, 9], 2),          # odd D everywhere: scalar / non-TMA paths
    (2, 2, [5, 3, 4, 3], 0),
    (2, 2, [6, 4, 5, 3], 3),
    (2, 2, [4, 3, 3, 2], 4),
    (2, 3, [6, 4, 5, 4, 3], 1),
    (3, 3, [4, 3, 5, 3, 4, 2], 1),
    (3, 3, [3, 2, 2, 3, 2, 2], 2),
    (2, 2, [1, 2, 1, 3], 1),          # single-cell axes
    (2, 2, [40, 33, 6, 5], 1),        # many lines per TMA tile + ragged last tile
]
KINDS_FRAC = ["small", "cfl", "edge"]
KINDS_INT = ["int0", "int+1", "int-1", "int+3", "int-3", "intwrap", "intmix"]


@pytest.mark.parametrize("geom", GEOMS, ids=lambda g: f"{g[0]}x{g[1]}v-{'x'.join(map(str, g[2]))}-k{g[3]}")
def test_every_axis_every_shift_kind(P, geom):
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k)
    f0 = W.random_field(o.shape, seed=W.SEED + k)
    for axis in range(dx + dv):
        n = o.D[dx + axis] if axis < dx else o.X
        for kind in KINDS_FRAC + KINDS_INT:
            delta = W.delta_table(n, kind, seed=W.SEED + axis, ncells=cells[axis]).numpy()
            want = o.sweep_axis(f0.numpy(), axis, delta)
            fg = f0.to(g.device).contiguous()
            g.advect_axis(fg, axis, delta)
            got = fg.cpu().numpy()
            if kind in KINDS_INT:
                assert np.array_equal(got, want), (axis, kind)
            else:
                assert rel_inf(got, want) <= TOL_SWEEP, (axis, kind, rel_inf(got, want))


def test_integer_shift_keeps_negative_zero_nan_and_inf(P):
    """alpha == 0 is a copy, not A=I,B=0 arithmetic: -0.0, inf and NaN payloads survive bit for bit."""
    g, o = make_pair(P, 2, 2, [6, 4, 4, 4], 1)
    f0 = W.random_field(o.shape, seed=5)
    f0.view(-1)[::7] = -0.0
    f0.view(-1)[3::11] = float("inf")
    f0.view(-1)[5::13] = float("nan")
    for axis in range(4):
        n = o.D[2 + axis] if axis < 2 else o.X
        delta = W.delta_table(n, "intmix", seed=3 + axis).numpy()
        want = o.sweep_axis(f0.numpy(), axis, delta)
        fg = f0.to(g.device).contiguous()
        g.advect_axis(fg, axis, delta)
        assert np.array_equal(fg.cpu().numpy().view(np.int64), want.view(np.int64))


@pytest.mark.parametrize("cells,k", [([9, 31, 4, 5], 1), ([7, 33, 3, 5], 2), ([64, 40, 3, 4], 2), ([5, 37, 2, 3], 0),
                                     ([1, 9, 2, 3], 1), ([3, 50, 3, 3], 4), ([700, 3, 2, 2], 3)])
def test_axis0_implementations_and_tilings_agree_bitwise(P, cells, k):
    """Every axis-0 kernel (per-warp TMA pipelines at every ring depth, block-wide TMA tiles, register walk) and
    every chunk size gives the same bits (same per-cell arithmetic), and matches the oracle."""
    g, o = make_pair(P, 2, 2, cells, k)
    f0 = W.random_field(o.shape, seed=9)
    delta = W.delta_table(o.D[2], "cfl", seed=1, ncells=cells[0]).numpy()
    outs = []
    for impl, stages in ((1, 1), (1, 2), (1, 3), (1, 4), (2, 1), (3, 1)):
        g.set_option("axis0_impl", impl)
        g.set_option("tile_stages", stages)
        for tb in (256, 1024, 4096, 16384, 65536):
            g.set_option("tile_bytes", tb)
            fg = f0.to(g.device).contiguous()
            g.advect_axis(fg, 0, delta)
            outs.append(fg.cpu().numpy())
    for x in outs[1:]:
        assert np.array_equal(outs[0], x)
    assert rel_inf(outs[0], o.sweep_axis(f0.numpy(), 0, delta)) <= TOL_SWEEP


# --------------------------------------------------------------- the named calls

def small_cfgs():
    c = W.CONFIGS
    return [c[0],
            W.scaled(c[1], [12, 10, 8, 8]),
            W.scaled(c[2], [8, 8, 6, 6, 4]),
            W.scaled(c[3], [6, 4, 4, 6, 4, 4]),
            W.scaled(c[4], [6, 4, 6, 4, 6, 4])]


@pytest.mark.parametrize("cfg", small_cfgs(), ids=lambda c: c["name"])
def test_advect_x_advect_v_density_poisson(P, cfg):
    g, o = pair_of_cfg(P, cfg)
    coords = [o.node_coords(a) for a in range(o.d)]
    f0 = W.random_field(o.shape, kind="perturbed", base=W.initial_data(cfg, coords))
    dt = cfg["dt"]
    # advect_x
    fg = f0.to(g.device).contiguous()
    g.advect_x(fg, dt / 2)
    want = o.advect_x(f0.numpy(), dt / 2)
    assert rel_inf(fg.cpu().numpy(), want) <= TOL_SWEEP * cfg["dim_x"]
    # density
    rho_g = g.density(fg).cpu().numpy()
    rho_o = o.density(want)
    assert rel_inf(rho_g, rho_o) <= 1e-12
    # poisson on the oracle's rho (same input both sides)
    E_g = g.poisson(torch.from_numpy(rho_o).to(g.device)).cpu().numpy()
    E_o = o.poisson(rho_o)
    assert rel_inf(E_g, E_o) <= 1e-12
    # advect_v with the physical field and with a strong random field (|delta| up to ~3 cells)
    hv = (cfg["domain"][2 * cfg["dim_x"] + 1] - cfg["domain"][2 * cfg["dim_x"]]) / cfg["cells"][cfg["dim_x"]]
    for E in (E_o, W.random_E(o.dx, o.xshape, amplitude=3.0 * hv / dt).numpy()):
        fg = f0.to(g.device).contiguous()
        g.advect_v(fg, torch.from_numpy(E).to(g.device), dt)
        want = o.advect_v(f0.numpy(), E, dt)
        assert rel_inf(fg.cpu().numpy(), want) <= TOL_SWEEP * cfg["dim_x"]


def test_advect_v_constant_dyadic_field_is_exact_integer_shift(P):
    """E = m h_v / dt with dyadic h_v, dt: delta = -m exactly -> bit-exact permutation through advect_v
    (the device-built shift table takes the same floor() decision as the oracle, in fp64)."""
    dom = [0, 1.0, 0, 1.0, -3.0, 3.0, -1.5, 1.5]
    g, o = make_pair(P, 2, 2, [4, 6, 8, 4], 1, dom)            # h_v = 0.75
    f0 = W.random_field(o.shape, seed=11)
    dt = 0.25
    E = np.empty((2,) + o.xshape)
    E[0] = 2 * 0.75 / dt
    E[1] = -1 * 0.75 / dt
    fg = f0.to(g.device).contiguous()
    g.advect_v(fg, torch.from_numpy(E).to(g.device), dt)
    want = o.advect_v(f0.numpy(), E, dt)
    assert np.array_equal(fg.cpu().numpy(), want)
    assert np.array_equal(want, np.roll(np.roll(f0.numpy(), -2 * 2, axis=1), 1 * 2, axis=0))


@pytest.mark.parametrize("cfg", small_cfgs(), ids=lambda c: c["name"])
def test_ten_strang_steps(P, cfg, parity_report):
    g, o = pair_of_cfg(P, cfg)
    coords = [o.node_coords(a) for a in range(o.d)]
    f0 = W.initial_data(cfg, coords)
    fg = f0.to(g.device).contiguous()
    fo = f0.numpy()
    m0 = g.mass(fg)
    for _ in range(10):
        g.step(fg, cfg["dt"])
        fo, rho_o, E_o = o.step(fo, cfg["dt"])
    assert parity_report.add("10 Strang steps", cfg["name"], "f", fg.cpu().numpy(), fo, TOL_STEPS) <= TOL_STEPS
    assert parity_report.add("10 Strang steps", cfg["name"], "rho of step 10", g.last_rho().cpu().numpy(), rho_o, TOL_STEPS) <= TOL_STEPS
    # E comes from rho - 1 (1e-2..1e-3 of rho), so relative to max|E| it carries rho's error times max|rho| / max|rho - 1|;
    # the stated relative bar still holds with two orders to spare (profiles/r2_parity.md)
    assert parity_report.add("10 Strang steps", cfg["name"], "E of step 10", g.last_E().cpu().numpy(), E_o, TOL_STEPS) <= TOL_STEPS
    assert abs(g.mass(fg) - m0) <= 1e-12 * abs(m0)
    assert abs(g.mass(fg) - o.mass(fo)) <= 1e-12 * abs(m0)
    Eg = g.last_E()
    assert abs(g.electric_energy(Eg) - o.electric_energy(Eg.cpu().numpy())) <= 1e-12 * o.electric_energy(E_o) + 1e-30


def next_cfgs():
    """the paper's bump-on-tail case (4th order) and CFL > 1 steps
    (PAPER.md:351-357), on grids the oracle finishes in seconds."""
    n = W.NEXT_CONFIGS
    b4 = n[0]
    return [b4, W.with_cfl(b4, 2.5), W.with_cfl(b4, 5.0),
            W.scaled(n[1], [4, 3, 4, 3, 2]), W.with_cfl(W.scaled(n[2], [3, 2, 2, 3, 2, 2]), 3.0)]


@pytest.mark.parametrize("cfg", next_cfgs(), ids=lambda c: c["name"])
def test_bump_on_tail_and_cfl_above_one_ten_strang_steps(P, cfg, parity_report):
    g, o = pair_of_cfg(P, cfg)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    fg, fo = f0.to(g.device).contiguous(), f0.numpy()
    m0 = g.mass(fg)
    for _ in range(10):
        g.step(fg, cfg["dt"])
        fo, rho_o, E_o = o.step(fo, cfg["dt"])
    assert parity_report.add("10 Strang steps (k = 3, CFL up to 5)", cfg["name"], "f", fg.cpu().numpy(), fo, TOL_STEPS) <= TOL_STEPS
    assert parity_report.add("10 Strang steps (k = 3, CFL up to 5)", cfg["name"], "E of step 10", g.last_E().cpu().numpy(), E_o,
                             TOL_STEPS) <= TOL_STEPS
    assert abs(g.mass(fg) - m0) <= 1e-12 * abs(m0)


def test_step_host_matches_step(P):
    cfg = W.CONFIGS[0]
    g, o = pair_of_cfg(P, cfg)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    fd = f0.to(g.device).contiguous()
    for _ in range(3):
        g.step(fd, cfg["dt"])
    fh = f0.clone().pin_memory()
    fdev = g.empty_field()
    Eh = torch.empty((2,) + o.xshape, dtype=torch.float64).pin_memory()
    g.step_host(fh, fdev, cfg["dt"], nsteps=3, E_host=Eh)
    assert torch.equal(fh, fd.cpu())
    assert torch.equal(Eh, g.last_E().cpu())


def test_errors_are_reported_not_swallowed(P):
    import ctypes as C
    L = P.lib()
    h = C.c_void_p()
    bad = L.sldg_create(C.byref(h), 3, 2, (C.c_int * 5)(2, 2, 2, 2, 2), 1, (C.c_double * 10)(*([0, 1] * 5)))
    assert bad == -1
    g, o = make_pair(P, 1, 1, [4, 4], 1)
    f = g.empty_field()
    assert L.sldg_step(None, C.c_void_p(f.data_ptr()), 0.1) == -1
    assert L.sldg_advect_x(g._h, None, 0.1) == -1
    assert L.sldg_advect_x(g._h, C.c_void_p(f.data_ptr() + 8), 0.1) == -1      # misaligned
    # a context without workspace refuses to run
    h2 = C.c_void_p()
    assert L.sldg_create(C.byref(h2), 1, 1, (C.c_int * 2)(4, 4), 1, (C.c_double * 4)(0, 1, 0, 1)) == 0
    assert L.sldg_step(h2, C.c_void_p(f.data_ptr()), 0.1) == -4
    L.sldg_destroy(h2)


# --------------------------------------------------------------- fused x1+x2 pass, in-place walks, step plans

FUSE_GEOMS = [
    (2, 2, [8, 8, 16, 16], 1),
    (2, 2, [7, 5, 6, 9], 2),
    (2, 2, [64, 9, 3, 4], 2),          # D_0 = 192: one plane per block
    (2, 2, [5, 37, 4, 3], 0),
    (2, 2, [3, 4, 3, 2], 4),
    (2, 2, [6, 5, 2, 3], 3),
    (2, 3, [6, 4, 5, 4, 3], 1),
    (3, 3, [4, 3, 5, 3, 4, 2], 1),
    (3, 3, [20, 7, 3, 2, 2, 2], 1),    # D_0 = 40: blocks straddle planes, ragged last block
    (2, 2, [1, 1, 2, 3], 1),
    (2, 2, [6, 1, 3, 2], 1),           # a single x_2 cell: the wrap cell is the only donor pair
    (2, 2, [64, 64, 1, 2], 2),         # BASELINE cfg2's x plane
    (2, 2, [100, 3, 2, 2], 2),         # D_0 = 300 > 256 threads: falls back to separate sweeps
]


@pytest.mark.parametrize("geom", FUSE_GEOMS, ids=lambda g: f"{g[0]}x{g[1]}v-{'x'.join(map(str, g[2]))}-k{g[3]}")
@pytest.mark.parametrize("tau", [0.013, 0.4, 7.7])
def test_advect_x_plans_agree_bitwise_and_match_oracle(P, geom, tau):
    """advect_x with the fused x1+x2 pass / separate sweeps, with and without in-place walks, and with fewer
    planes per block: identical bits (same per-value arithmetic in the same order), and parity with the oracle.
    tau = 0.013: |delta| < 1 everywhere (in-place walks allowed); 7.7: CFL > 1 (they are not)."""
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k)
    f0 = W.random_field(o.shape, seed=21 + k)
    outs = []
    # (fuse_x, inplace_walk, fused_threads, fused_impl, cell_rows, cell_threads, cell_stages, x_copy)
    # x_copy = 1: the plan of the other buffer parity + one copy (for dim_x = 2 the fused pass runs only there)
    plans = ((1, 1, 256, 0, 0, 128, 3, 0), (1, 0, 256, 0, 0, 128, 3, 0), (0, 1, 256, 0, 0, 128, 3, 0),
             (0, 0, 256, 0, 0, 128, 3, 0), (0, 0, 256, 0, 0, 128, 3, 1), (1, 1, 256, 0, 0, 128, 3, 1),
             (1, 1, 256, 2, 0, 128, 3, 0), (1, 1, 64, 2, 0, 128, 3, 1), (1, 1, 256, 2, 0, 128, 3, 1),     # node-per-thread fused kernel
             (1, 1, 256, 1, 1, 128, 2, 0), (1, 1, 256, 1, 1, 128, 2, 1), (1, 1, 256, 1, 3, 64, 3, 1),     # cell-per-thread fused kernel
             (1, 1, 256, 1, 5, 96, 4, 1), (1, 1, 256, 1, 64, 32, 6, 1))
    for fuse, inplace, threads, impl, rows, cthreads, cstages, xcopy in plans:
        g.set_option("fuse_x", fuse); g.set_option("inplace_walk", inplace); g.set_option("fused_threads", threads)
        g.set_option("x_copy", xcopy)
        g.set_option("fused_impl", impl); g.set_option("cell_rows", rows); g.set_option("cell_threads", cthreads)
        g.set_option("cell_stages", cstages)
        fg = f0.to(g.device).contiguous()
        g.advect_x(fg, tau)
        outs.append(fg.cpu().numpy())
    for x in outs[1:]:
        assert np.array_equal(outs[0], x)
    assert rel_inf(outs[0], o.advect_x(f0.numpy(), tau)) <= TOL_SWEEP * dx


def test_advect_x_integer_shifts_are_exact_in_every_plan(P):
    """v nodes chosen so that v*tau/h_x is an integer on every line: the fused pass copies, bit for bit."""
    # h_x = 0.25 on both x axes; v nodes of a k=0 grid on [-4,4] with 8 cells: -3.5..3.5; tau = 0.5 -> delta = 2 v
    dom = [0, 1.0, 0, 1.5, -4.0, 4.0, -4.0, 4.0]
    g, o = make_pair(P, 2, 2, [4, 6, 8, 8], 0, dom)
    f0 = W.random_field(o.shape, seed=4)
    f0.view(-1)[::5] = -0.0
    want = o.advect_x(f0.numpy(), 0.5)
    for fuse, impl, xcopy in ((1, 0, 0), (1, 0, 1), (1, 1, 1), (1, 2, 1), (0, 0, 0)):
        g.set_option("fuse_x", fuse); g.set_option("fused_impl", impl); g.set_option("x_copy", xcopy)
        fg = f0.to(g.device).contiguous()
        g.advect_x(fg, 0.5)
        assert np.array_equal(fg.cpu().numpy().view(np.int64), want.view(np.int64))


@pytest.mark.parametrize("cfg", small_cfgs()[1:], ids=lambda c: c["name"])
def test_step_plans_agree_bitwise(P, cfg):
    g, o = pair_of_cfg(P, cfg)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    outs = []
    for fuse, inplace, impl in ((1, 1, 0), (1, 0, 0), (0, 1, 0), (0, 0, 0), (1, 1, 2)):
        g.set_option("fuse_x", fuse); g.set_option("inplace_walk", inplace); g.set_option("fused_impl", impl)
        fg = f0.to(g.device).contiguous()
        for _ in range(3):
            g.step(fg, cfg["dt"])
        outs.append(fg.cpu().numpy())
    for x in outs[1:]:
        assert np.array_equal(outs[0], x)


# --------------------------------------------------------------- CUDA graph replay of the Strang step

@pytest.mark.parametrize("cfg", [small_cfgs()[0], small_cfgs()[3]], ids=lambda c: c["name"])
def test_graph_replay_of_the_step_is_bitwise_the_plain_step(P, cfg):
    """Small problems replay a captured CUDA graph (launch-latency bound): same kernels,
    same order, same bits; the graph is rebuilt when dt changes or when another call rewrites the x-sweep tables."""
    g, o = pair_of_cfg(P, cfg)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    dt = cfg["dt"]
    seq = [dt, dt, dt, 0.5 * dt, 0.5 * dt, dt]
    outs = []
    for graph in (0, 2, 1):
        g.set_option("graph", graph)
        fg = f0.to(g.device).contiguous()
        n0 = g.launch_count()
        for i, h in enumerate(seq):
            g.step(fg, h)
            # the replay path is really taken (the binding hands over torch's default stream, on which a capture cannot
            # start: the library then records on a stream of its own), and never with graph = 0
            assert g.graph_active() == (graph != 0), (graph, i)
            if i == 1:
                g.advect_x(fg, 0.3 * dt)            # rewrites the cached x tables: the graph must not survive
                assert not g.graph_active()
        outs.append((fg.cpu().numpy(), g.launch_count() - n0))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][0], outs[2][0])
    assert outs[0][1] == outs[1][1] == outs[2][1]                 # replays count the launches they contain
    fo = f0.numpy()
    for i, h in enumerate(seq):
        fo, _, _ = o.step(fo, h)
        if i == 1:
            fo = o.advect_x(fo, 0.3 * dt)
    assert rel_inf(outs[0][0], fo) <= TOL_STEPS


def test_contexts_of_different_degree_live_side_by_side(P):
    """The A/B polynomial coefficients of the device-side v-table kernel are per context: a k=1 context keeps working
    after a k=2 (and a k=3) context was created on the same device (they used to share one __constant__ copy)."""
    dom = [0.0, 4 * np.pi, 0.0, 4 * np.pi, -6.0, 6.0, -6.0, 6.0]
    cells = [4, 4, 6, 6]
    ctxs = {}
    for k in (1, 2, 3, 1):                               # the second k=1 context is created last
        ctxs.setdefault(k, []).append((P.Sldg(2, 2, cells, k, dom), O.Oracle(2, 2, cells, k, dom)))
    for k in (1, 2, 3):
        for g, o in ctxs[k]:
            rng = np.random.default_rng(W.SEED + k)
            f0 = rng.random(tuple(reversed(o.D)))
            E = rng.uniform(-3.0, 3.0, size=(2,) + tuple(reversed(o.D[:2])))
            fg = torch.from_numpy(f0).to(g.device).contiguous()
            g.advect_v(fg, torch.from_numpy(E).to(g.device).contiguous(), 0.37)
            want = o.advect_v(f0, E, 0.37)
            assert rel_inf(fg.cpu().numpy(), want) <= 1e-12, k


# --------------------------------------------------------------- fused x1+x2+x3 pass (dim_x = 3, degree <= 1)

F3_GEOMS = [
    (3, 3, [4, 3, 5, 3, 4, 2], 1),
    (3, 3, [20, 7, 3, 2, 2, 2], 1),    # D_0 = 40 as in BASELINE cfg4; 7 x_2 cells: ragged strips
    (3, 3, [6, 5, 1, 2, 3, 2], 1),     # a single x_3 cell: the wrap cell is the only donor pair
    (3, 3, [4, 1, 3, 2, 2, 3], 1),     # a single x_2 cell: halo = the cell itself
    (3, 3, [8, 6, 4, 2, 3, 2], 0),     # degree 0 (D_0 = 8: bulk-copy rule holds)
    (3, 3, [5, 4, 3, 2, 2, 2], 0),     # degree 0, D_0 = 5: rows not a multiple of 16 B -> planner falls back
]


@pytest.mark.parametrize("geom", F3_GEOMS, ids=lambda g: f"{'x'.join(map(str, g[2]))}-k{g[3]}")
@pytest.mark.parametrize("tau", [0.013, 0.4, 7.7])
def test_fused3_pass_agrees_bitwise_with_separate_sweeps_and_matches_oracle(P, geom, tau):
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k)
    f0 = W.random_field(o.shape, seed=31 + k)
    outs = []
    # (fuse3, fuse_x, x_copy, f3_threads, f3_stages)
    for fuse3, fuse, xcopy, thr, st in ((0, 0, 0, 128, 2), (0, 1, 0, 128, 2), (1, 1, 1, 128, 2), (1, 1, 1, 256, 3),
                                        (1, 1, 1, 24, 4), (1, 1, 1, 1, 2)):
        g.set_option("fuse3", fuse3); g.set_option("fuse_x", fuse); g.set_option("x_copy", xcopy)
        g.set_option("f3_threads", thr); g.set_option("f3_stages", st)
        fg = f0.to(g.device).contiguous()
        g.advect_x(fg, tau)
        outs.append(fg.cpu().numpy())
    for x in outs[1:]:
        assert np.array_equal(outs[0], x)
    assert rel_inf(outs[0], o.advect_x(f0.numpy(), tau)) <= TOL_SWEEP * dx


def test_fused3_integer_shifts_are_exact(P):
    dom = [0, 1.0, 0, 1.5, 0, 0.5, -4.0, 4.0, -4.0, 4.0, -4.0, 4.0]
    g, o = make_pair(P, 3, 3, [4, 6, 2, 8, 8, 8], 0, dom)          # h_x = 0.25; v nodes -3.5..3.5; tau 0.5 -> delta = 2 v
    f0 = W.random_field(o.shape, seed=4)
    f0.view(-1)[::5] = -0.0
    want = o.advect_x(f0.numpy(), 0.5)
    for fuse3 in (1, 0):
        g.set_option("fuse3", fuse3); g.set_option("x_copy", 1)
        fg = f0.to(g.device).contiguous()
        g.advect_x(fg, 0.5)
        assert np.array_equal(fg.cpu().numpy().view(np.int64), want.view(np.int64))


@pytest.mark.parametrize("cfg", small_cfgs()[3:], ids=lambda c: c["name"])
def test_step_with_and_without_fused3_agree_bitwise(P, cfg):
    g, o = pair_of_cfg(P, cfg)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    outs = []
    for fuse3 in (1, 0):
        g.set_option("fuse3", fuse3)
        fg = f0.to(g.device).contiguous()
        n0 = g.launch_count()
        for _ in range(3):
            g.step(fg, cfg["dt"])
        outs.append((fg.cpu().numpy(), g.launch_count() - n0))
    assert np.array_equal(outs[0][0], outs[1][0])
    assert outs[0][1] < outs[1][1]                                  # the fused plan really ran (fewer launches)


@pytest.mark.parametrize("cfg", [small_cfgs()[1], small_cfgs()[3], small_cfgs()[4]], ids=lambda c: c["name"])
@pytest.mark.parametrize("n", [1, 2, 3, 4])
@pytest.mark.parametrize("fuse_v", [0, 2])
def test_steps_equals_repeated_step_bitwise(P, cfg, n, fuse_v):
    """sldg_steps may alternate buffers between steps: same bits, result in f.  It saves passes exactly when a single
    step, which must end in f, cannot use its one-pass plans: dim_x = 3 with three separate v sweeps (odd flips: only one
    of the two x half steps can be the fused x_1+x_2+x_3 pass), dim_x = 2 with the fused v_1+v_2 pass (odd flips again).
    fuse_v = 2: these small grids are below the auto rule's size."""
    g, o = pair_of_cfg(P, cfg)
    g.set_option("graph", 0)
    g.set_option("fuse_v", fuse_v)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    fa, fb = f0.to(g.device).contiguous(), f0.to(g.device).contiguous()
    n0 = g.launch_count()
    for _ in range(n):
        g.step(fa, cfg["dt"])
    n1 = g.launch_count()
    g.steps(fb, cfg["dt"], n)
    n2 = g.launch_count()
    assert torch.equal(fa, fb)
    odd_v_flips = (cfg["dim_x"] == 3) == (fuse_v == 0)
    # dim_x = 2: sldg_steps also merges the x half steps of consecutive steps into one pass (tests/test_gpu_xdouble.py)
    merged = cfg["dim_x"] == 2 and (n >= 3 or (n == 2 and fuse_v == 2))
    if (odd_v_flips and n >= 2) or merged:
        assert n2 - n1 < n1 - n0                                    # fewer passes
    else:
        assert n2 - n1 == n1 - n0


# --------------------------------------------------------------- determinism under load (race detector of last resort)

@pytest.mark.parametrize("geom,prec", [((2, 2, [48, 40, 12, 10], 2), "f64"), ((3, 3, [12, 10, 12, 6, 5, 4], 1), "f64"),
                                       ((2, 2, [32, 32, 16, 12], 3), "f64"), ((3, 3, [12, 10, 12, 6, 5, 4], 1), "f32"),
                                       ((2, 3, [32, 24, 8, 8, 6], 1), "f32")],
                         ids=lambda v: v if isinstance(v, str) else "x".join(map(str, v[2])) + f"-k{v[3]}")
def test_repeated_steps_are_bitwise_identical(P, geom, prec):
    """Grids large enough to fill every SM several times: 6 runs of 3 Strang steps (fused passes, TMA rings, bulk
    stores, in-place walks) from the same data give the same bits; a missing barrier or fence would not."""
    dx, dv, cells, k = geom
    dom = []
    for a in range(dx + dv):
        dom += [0.0, 4 * math.pi] if a < dx else [-6.0, 6.0]
    g = P.Sldg(dx, dv, cells, k, dom, precision=prec)
    g.set_option("graph", 0)
    f0 = W.random_field(g.shape, seed=77, device=g.device).to(g.dtype)
    ref = None
    for rep in range(6):
        f = f0.clone()
        g.steps(f, 0.1, 3)
        if ref is None:
            ref = f
        else:
            assert torch.equal(ref, f), rep


# --------------------------------------------------------------- single-launch Poisson solve of small x grids

@pytest.mark.parametrize("geom", [(1, 1, [37, 5], 1), (2, 2, [8, 8, 4, 4], 1), (2, 2, [7, 5, 3, 3], 2), (2, 3, [6, 4, 3, 2, 2], 3),
                                  (3, 3, [4, 3, 5, 2, 2, 2], 1), (3, 3, [3, 3, 2, 2, 2, 2], 2), (2, 2, [16, 16, 2, 2], 1)],
                         ids=lambda g: f"{g[0]}x{g[1]}v-{'x'.join(map(str, g[2]))}-k{g[3]}")
def test_small_grid_poisson_in_one_launch_is_bitwise_the_multi_launch_route(P, geom):
    """X <= 1024 x nodes (BASELINE config 1: 256): one single-block launch with the work arrays in shared memory does the
    per-axis DFTs, the spectral solve and the inverse transforms with the same fma chain per output as the tiled
    kernels: same bits, 1 launch instead of 8 / 15; and the oracle's E within the bar."""
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k)
    rho = 1.0 + 0.3 * W.random_field(o.xshape, seed=8)
    outs = []
    for small in (1, 0):
        g.set_option("poisson_small", small)
        n0 = g.launch_count()
        E = g.poisson(rho.to(g.device))
        outs.append((E.cpu().numpy(), g.launch_count() - n0))
    assert np.array_equal(outs[0][0], outs[1][0])
    assert outs[0][1] == 1 and outs[1][1] == dx + dx * (1 + dx)
    assert rel_inf(outs[0][0], o.poisson(rho.numpy())) <= 1e-12


# --------------------------------------------------------------- boundary behaviour (include/sldg.h)

def test_x_table_cache_holds_two_time_increments(P):
    """include/sldg.h STREAM / SYNC: the x-sweep tables of two time increments stay cached per axis, so a caller that
    alternates advect_x(dt) and advect_x(dt/2) uploads (and synchronises) only in the first two calls; a third
    increment evicts the least recently used one."""
    g, o = make_pair(P, 2, 2, [6, 5, 4, 3], 1)
    f = W.random_field(o.shape, seed=5).to(g.device).contiguous()
    g.timing_enable(True); g.timing_read()
    g.advect_x(f, 0.1); g.advect_x(f, 0.05)
    kinds, _ = g.timing_read()
    assert kinds["table_uploads"][0] == 2 * 2                       # two increments x two axes, one upload event each
    for _ in range(3):
        g.advect_x(f, 0.1); g.advect_x(f, 0.05)
    kinds, _ = g.timing_read()
    assert kinds["table_uploads"][0] == 0                           # cached: no upload, no synchronisation
    g.advect_x(f, 0.2); g.advect_x(f, 0.05); g.advect_x(f, 0.2)
    kinds, _ = g.timing_read()
    assert kinds["table_uploads"][0] == 2                           # 0.2 evicted 0.1 (least recently used); 0.05 stayed
    g.advect_x(f, 0.1)
    kinds, _ = g.timing_read()
    assert kinds["table_uploads"][0] == 2
    g.timing_enable(False)


def test_non_finite_time_increment_and_shifts_are_rejected(P):
    g, o = make_pair(P, 2, 2, [6, 5, 4, 3], 1)
    f0 = W.random_field(o.shape, seed=5)
    f = f0.to(g.device).contiguous()
    for bad in (float("nan"), float("inf"), -float("inf")):
        with pytest.raises(P.SldgError, match="invalid argument"):
            g.advect_x(f, bad)
        with pytest.raises(P.SldgError, match="invalid argument"):
            g.step(f, bad)
        d = np.zeros(o.D[2]); d[3] = bad
        with pytest.raises(P.SldgError, match="invalid argument"):
            g.advect_axis(f, 0, d)
        d = np.zeros(o.X); d[7] = bad
        with pytest.raises(P.SldgError, match="invalid argument"):
            g.advect_axis(f, 2, d)
    assert torch.equal(f.cpu(), f0)                          # nothing was enqueued


@pytest.mark.parametrize("geom", [(2, 2, [8, 6, 6, 5], 1), (3, 3, [4, 3, 2, 4, 3, 2], 1), (2, 3, [6, 4, 5, 4, 3], 2)],
                         ids=lambda g: f"{g[0]}x{g[1]}v-k{g[3]}")
def test_declined_fused_passes_fall_back_to_the_same_bits(P, geom):
    """include/sldg.h: a fused pass whose launcher declines (cudaErrorNotSupported) is replaced by the separate sweeps,
    plus one device copy where the buffer parity differs -- same bits, never an error (test knob `decline`)."""
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k)
    f0 = W.random_field(o.shape, seed=8)
    outs = []
    for decline in (0, 1, 2, 4, 8, 16, 31):
        g.set_option("graph", 0); g.set_option("fuse_v", 2); g.set_option("fuse_v3", 2); g.set_option("x_double", 2)
        g.set_option("decline", decline)
        fg = f0.to(g.device).contiguous()
        g.steps(fg, 0.07, 3)
        g.step(fg, 0.07)
        E = g.last_E()
        g.advect_v(fg, E, 0.07)
        g.advect_x(fg, 0.07)
        outs.append(fg.cpu().numpy())
    for x in outs[1:]:
        assert np.array_equal(outs[0], x)


@pytest.mark.parametrize("rho_by", ["second context", "density_static"])
def test_v_shard_plumbing_drives_the_cuda_context(P, rho_by):
    """paper_2110_14557_b200/shard.py with the CUDA context as its engine (single rank: the halo exchange is the periodic
    wrap of the rank's own slab): a context on the widened sub-domain for the sweeps, one on the interior for rho.  The
    interior must equal the plain single-domain steps (same sweeps; rho summed over the same values in another order).
    "density_static": rho of the interior through the context-free entry point instead of a second context (and workspace)."""
    from paper_2110_14557_b200 import shard as S
    cfg = W.scaled(W.CONFIGS[0], [6, 4, 6, 8])
    g, o = pair_of_cfg(P, cfg)
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)])
    ref = f0.to(g.device).contiguous()
    for _ in range(3):
        g.step(ref, cfg["dt"])
    geom = S.Geometry(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
    H = 2
    make = lambda gm: P.Sldg(gm.dim_x, gm.dim_v, gm.cells, gm.degree, gm.domain)
    sh = S.VShard(geom, 0, 1, H, make)
    if rho_by == "density_static":
        sh = S.VShard(geom, 0, 1, H, make, interior_density=S.cuda_interior_density(P, sh.interior))
        assert sh.eng_int is None
    k1 = cfg["degree"] + 1
    f_ext = torch.zeros(tuple(reversed([c * k1 for c in sh.extended.cells])), dtype=torch.float64, device=g.device)
    sh.interior_of(f_ext).copy_(f0)
    for _ in range(3):
        sh.step(f_ext, cfg["dt"])
    got, want = sh.interior_of(f_ext).cpu().numpy(), ref.cpu().numpy()
    assert rel_inf(got, want) <= 1e-13


@pytest.mark.parametrize("geom", [(2, 2, [32, 32, 16, 16], 1), (2, 2, [21, 14, 12, 8], 2), (2, 3, [16, 10, 6, 6, 5], 1)],
                         ids=lambda g: f"{g[0]}x{g[1]}v-{'x'.join(map(str, g[2]))}-k{g[3]}")
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_density_through_tensor_copies_matches_plain_loads_and_the_oracle(P, geom, prec, parity_report):
    """Row a3 on problems large enough for the TMA kernel (x tiles x v chunks >= 2 per SM; ragged last x tile and last box):
    both kernels against the oracle at the per-operation bar, each of them bitwise reproducible, and really different launches."""
    dx, dv, cells, k = geom
    dom = []
    for a in range(dx + dv):
        dom += [0.0, 1.0 + a] if a < dx else [-2.0 - a, 2.0 + a]
    g = P.Sldg(dx, dv, cells, k, dom, precision=prec)
    o = O.Oracle(dx, dv, cells, k, dom, threads=O.lib().orc_max_threads())
    f0 = W.random_field(o.shape, seed=31)
    if prec == "f32":
        f0 = f0.to(torch.float32)
    fg = f0.to(g.device).contiguous()
    want = o.density(f0.numpy()) if prec == "f64" else o.density_f32(f0.numpy())
    outs = []
    for tma in (1, 0, 1):
        g.set_option("rho_tma", tma)
        outs.append(g.density(fg).cpu().numpy())
    assert np.array_equal(outs[0], outs[2])                              # deterministic
    for name, r in (("tensor copies", outs[0]), ("plain loads", outs[1])):
        assert parity_report.add("density, " + name, "x".join(map(str, cells)) + f" k={k}", "rho", r, want, TOL_SWEEP, prec) <= TOL_SWEEP
    # the two kernels chunk the v sum differently: they may differ, but only by the rounding of two fp64 sums of <= 1024 terms
    assert rel_inf(outs[0], outs[1]) <= 1e-14
