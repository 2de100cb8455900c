"""GPU parity at BASELINE.json's FULL sizes (configs 2-5), in the launch configuration bench.py times.

The oracle cannot hold 10-57 GB arrays, but every operation of the path decouples: x-sweeps act on x-space for a
fixed velocity node, v-sweeps and the density on v-space for a fixed x node.  So the test gathers, from the
full-size device array, the complete x-space of a few velocity CELLS and the complete v-space of a few x CELLS,
runs the full-size GPU call, and compares those slabs with the oracle applied to the same slabs as a small problem
(one cell per frozen axis).  Poisson runs on the full-size rho directly.  Single sweeps with random shift tables
(CFL > 1 and integer) are checked on sampled lines with the oracle's line routine.
Bars as in test_gpu_parity.py: 1e-12 per sweep, bit-exact for integer shifts.  The same slab / line tests run in single
precision mode (reading W) against the fp32 oracle (2e-6 per sweep, bit-exact integer shifts) on configs
2-5, and in fp64 on the paper's fourth-order bump-on-tail workloads (k = 3).  Every comparison appends
its measured error (max|g-o|/max|o| and the element-wise figure of reading L) to the parity report (conftest.py).
"""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import oracle as O

pytestmark = pytest.mark.gpu

TOL = 1e-12
TOL32 = 2e-6          # (2(k+1)+1) ulp32 of sum|A||u|, FMA chains against separately rounded products (reading W)


def rel_inf(g, o):
    return float(np.abs(g - o).max() / np.abs(o).max())


@pytest.fixture(scope="module")
def P():
    import paper_2110_14557_b200 as pkg
    if not torch.cuda.is_available():
        pytest.fail("gpu test without a CUDA device")
    return pkg


def cell_samples(cells, n, seed):
    """n seeded cell multi-indices, always including the first and the last cell."""
    rng = np.random.default_rng(seed)
    out = [tuple(0 for _ in cells), tuple(c - 1 for c in cells)]
    while len(out) < n:
        out.append(tuple(int(rng.integers(0, c)) for c in cells))
    return out


def slab_index(g, fixed_axes, cell):
    """Index tuple (torch dims are reversed axes) selecting all nodes of `cell` on `fixed_axes`, all else."""
    k1 = g.k + 1
    idx = [slice(None)] * g.d
    for a, i in zip(fixed_axes, cell):
        idx[g.d - 1 - a] = slice(i * k1, (i + 1) * k1)
    return tuple(idx)


def cell_domain(cfg, axis, i):
    lo, hi = cfg["domain"][2 * axis], cfg["domain"][2 * axis + 1]
    h = (hi - lo) / cfg["cells"][axis]
    return [lo + i * h, lo + (i + 1) * h]


ALL = {c["name"]: c for c in W.CONFIGS + W.NEXT_CONFIGS}
FULL_CASES = ([(W.CONFIGS[i]["name"], "f64") for i in (1, 2, 3, 4)] + [(W.CONFIGS[i]["name"], "f32") for i in (1, 2, 3, 4)] +
              [("bot_5d_k3_16", "f64"), ("bot_6d_k3_9", "f64")])


class Full:
    """One full-size problem on the device plus the oracle's functions of its precision."""

    def __init__(self, cfg, g, f, prec):
        self.cfg, self.g, self.f, self.prec = cfg, g, f, prec
        self.tol = TOL if prec == "f64" else TOL32
        self.np_dtype = np.float64 if prec == "f64" else np.float32

    def o_advect_x(self, o, b, tau):
        return o.advect_x(b, tau) if self.prec == "f64" else o.advect_x_f32(b, tau)

    def o_advect_v(self, o, b, E, tau):
        return o.advect_v(b, E, tau) if self.prec == "f64" else o.advect_v_f32(b, E, tau)

    def o_density(self, o, b):
        return o.density(b) if self.prec == "f64" else o.density_f32(b)

    def mass_tol(self):
        return 1e-12 if self.prec == "f64" else 2e-6


@pytest.fixture(scope="module", params=FULL_CASES, ids=lambda c: f"{c[0]}-{c[1]}")
def full(request, P):
    name, prec = request.param
    cfg = ALL[name]
    es = 8 if prec == "f64" else 4
    need = 2 * W.field_elems(cfg) * es + (6 << 30)
    free, _ = torch.cuda.mem_get_info()
    if free < need:
        pytest.fail(f"{cfg['name']}: needs {need >> 30} GiB of device memory, {free >> 30} GiB free")
    g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], precision=prec)
    f = g.empty_field()
    coords = [g.node_coords(a) for a in range(g.d)]
    if prec == "f32":                     # the generator works in fp64: fill slab by slab along the slowest axis
        D = f.shape[0]
        step = max(1, D // 8)
        for a in range(0, D, step):
            b = min(D, a + step)
            f[a:b].copy_(W.initial_data(cfg, coords[:-1] + [coords[-1][a:b]], device=g.device))
    else:
        W.initial_data(cfg, coords, device=g.device, out=f)
    W.perturb_inplace(f, seed=W.SEED + len(name))
    yield Full(cfg, g, f, prec)
    g.close()
    del f
    torch.cuda.empty_cache()


@pytest.mark.parametrize("xcopy", [0, 1], ids=["even-parity plan", "odd-parity plan (the one-pass fused sweeps)"])
def test_advect_x_on_full_x_space_of_sampled_velocity_cells(full, xcopy, parity_report):
    """x_copy = 1 runs the plan sldg_step / sldg_steps use for their flipping x half steps: the fused x1+x2 pass
    (dim_x = 2) or the fused x1+x2+x3 pass (dim_x = 3), in the launch configuration bench.py times."""
    cfg, g, f = full.cfg, full.g, full.f
    g.set_option("x_copy", xcopy)
    dx, dv = cfg["dim_x"], cfg["dim_v"]
    vaxes = list(range(dx, dx + dv))
    cells = cell_samples(cfg["cells"][dx:], 5, seed=1)
    before = [f[slab_index(g, vaxes, c)].cpu().numpy() for c in cells]
    tau = cfg["dt"] / 2
    m0 = g.mass(f)
    g.advect_x(f, tau)
    assert abs(g.mass(f) - m0) <= full.mass_tol() * abs(m0)
    for c, b in zip(cells, before):
        dom = list(cfg["domain"][:2 * dx])
        for a, i in zip(vaxes, c):
            dom += cell_domain(cfg, a, i)
        o = O.Oracle(dx, dv, cfg["cells"][:dx] + [1] * dv, cfg["degree"], dom, threads=O.lib().orc_max_threads())
        want = full.o_advect_x(o, b, tau)
        got = f[slab_index(g, vaxes, c)].cpu().numpy()
        err = parity_report.add("advect_x full x-space of a v cell", cfg["name"], f"x_copy={xcopy} v-cell {c}", got, want,
                                full.tol * dx, full.prec)
        assert err <= full.tol * dx, (c, err)
    g.set_option("x_copy", 0)


def test_density_poisson_advect_v_on_full_v_space_of_sampled_x_cells(full, parity_report):
    cfg, g, f = full.cfg, full.g, full.f
    dx, dv = cfg["dim_x"], cfg["dim_v"]
    xaxes = list(range(dx))
    cells = cell_samples(cfg["cells"][:dx], 5, seed=2)
    smalls = []
    for c in cells:
        dom = []
        for a, i in zip(xaxes, c):
            dom += cell_domain(cfg, a, i)
        dom += list(cfg["domain"][2 * dx:])
        smalls.append(O.Oracle(dx, dv, [1] * dx + cfg["cells"][dx:], cfg["degree"], dom,
                               threads=O.lib().orc_max_threads()))
    before = [f[slab_index(g, xaxes, c)].cpu().numpy() for c in cells]
    # density: full-size kernel vs the oracle on each sampled x cell
    rho = g.density(f)
    rho_h = rho.cpu().numpy()
    k1 = cfg["degree"] + 1
    xsl = [tuple(slice(i * k1, (i + 1) * k1) for i in reversed(c)) for c in cells]
    scale = np.abs(rho_h).max()
    for o, b, sl, c in zip(smalls, before, xsl, cells):
        want = full.o_density(o, b)
        parity_report.add("density of an x cell (scaled by max rho)", cfg["name"], f"x-cell {c}", rho_h[sl] / scale, want / scale,
                          TOL, full.prec)
        assert np.abs(rho_h[sl] - want).max() <= TOL * scale
    # Poisson on the full-size rho (the oracle's naive DFT handles X <= 110592)
    ofull = O.Oracle(dx, dv, cfg["cells"][:dx] + [1] * dv, cfg["degree"],
                     list(cfg["domain"][:2 * dx]) + [0.0, 1.0] * dv, threads=O.lib().orc_max_threads())
    E = g.poisson(rho)
    E_h = E.cpu().numpy()
    E_o = ofull.poisson(rho_h)
    # the stated per-operation bar, also on the largest x grids (measured: at most 5.2e-13, profiles/r2_parity.md)
    err = parity_report.add("poisson on the full-size rho", cfg["name"], f"X={g.X}", E_h, E_o, TOL, full.prec)
    assert err <= TOL, err
    # advect_v with the physical field and with a strong seeded field (|delta| up to ~3 cells)
    hv = (cfg["domain"][2 * dx + 1] - cfg["domain"][2 * dx]) / cfg["cells"][dx]
    dt = cfg["dt"]
    strong = W.random_E(dx, g.xshape, amplitude=3.0 * hv / dt, device=g.device)
    # second run: every fused v pass the shape allows, forced (dim_x = 3: the one-pass v_1+v_2+v_3 sweep that sldg_steps plans)
    for Efield, force in ((E, 1), (strong, 2)):
        Eh = Efield.cpu().numpy()
        m0 = g.mass(f)
        g.set_option("fuse_v", force); g.set_option("fuse_v3", force)
        g.advect_v(f, Efield, dt)
        g.set_option("fuse_v", 1); g.set_option("fuse_v3", 1)
        assert abs(g.mass(f) - m0) <= full.mass_tol() * abs(m0)
        after = []
        for o, b, c, sl in zip(smalls, before, cells, xsl):
            want = full.o_advect_v(o, b, np.ascontiguousarray(Eh[(slice(None),) + sl]), dt)
            got = f[slab_index(g, xaxes, c)].cpu().numpy()
            err = parity_report.add("advect_v full v-space of an x cell", cfg["name"],
                                    f"{'physical E' if force == 1 else 'strong seeded E, fused passes forced'} x-cell {c}", got, want,
                                    full.tol * dx, full.prec)
            assert err <= full.tol * dx, (c, err)
            after.append(got)
        before = after


@pytest.mark.parametrize("kind", ["cfl", "intmix"])
def test_single_sweeps_on_sampled_lines(full, kind, parity_report):
    """Every swept axis through the test hook at full size; 4092 seeded lines per axis against orc_sweep_line (fp32: the
    lines as a 1x1v problem through orc_sweep_axis_f32, one shift per line)."""
    cfg, g, f = full.cfg, full.g, full.f
    dx = cfg["dim_x"]
    k = cfg["degree"]
    rng = np.random.default_rng(7)
    for axis in range(2 * dx):
        Da = g.D[axis]
        inner = int(np.prod(g.D[:axis], dtype=np.int64)) if axis else 1
        outer = g.nf // (inner * Da)
        n = g.D[dx + axis] if axis < dx else g.X
        delta = W.delta_table(n, kind, seed=W.SEED + axis, ncells=cfg["cells"][axis]).numpy()
        ns = 4092                      # divisible by k+1 = 1..4
        q = np.concatenate([[0, outer - 1], rng.integers(0, outer, ns - 2)])
        p = np.concatenate([[0, inner - 1], rng.integers(0, inner, ns - 2)])
        qt, pt = torch.from_numpy(q).to(g.device), torch.from_numpy(p).to(g.device)
        f3 = f.view(outer, Da, inner)
        lines_in = f3[qt, :, pt].cpu().numpy()
        g.advect_axis(f, axis, delta)
        lines_out = f.view(outer, Da, inner)[qt, :, pt].cpu().numpy()
        if axis < dx:          # shift index = node of v-axis dx+axis = a digit of the outer index
            sdiv = int(np.prod(g.D[axis + 1:dx + axis], dtype=np.int64)) if dx + axis > axis + 1 else 1
            sidx = (q // sdiv) % g.D[dx + axis]
        else:                  # shift index = flat x node
            sidx = p % g.X
        if full.prec == "f64":
            want = np.stack([O.sweep_line(k, lines_in[i], delta[sidx[i]]) for i in range(ns)])
        else:
            ol = O.Oracle(1, 1, [cfg["cells"][axis], ns // (k + 1)], k, [0.0, 1.0, 0.0, 1.0], threads=O.lib().orc_max_threads())
            want = ol.sweep_axis_f32(lines_in, 0, delta[sidx])
        if kind == "intmix":
            assert np.array_equal(lines_out, want), axis
        else:
            err = parity_report.add("single sweep on 4092 sampled lines", cfg["name"], f"axis {axis}, CFL > 1 shifts", lines_out, want,
                                    full.tol, full.prec)
            assert err <= full.tol, (axis, err)


def test_constants_are_preserved_by_two_steps_at_full_size(full):
    """rows of A + B sum to 1 (invariant p4), so a constant f stays constant to round-off through
    every sweep of sldg_steps at full size (fused passes, in-place walks, v sweeps with E = 0 up to round-off).
    Runs last: it overwrites the module's f."""
    cfg, g, f = full.cfg, full.g, full.f
    f.fill_(0.375)
    g.steps(f, cfg["dt"], 2)
    lo, hi = float(f.min()), float(f.max())
    bar = 1e-13 if full.prec == "f64" else 2e-6
    assert abs(lo - 0.375) <= bar and abs(hi - 0.375) <= bar, (lo, hi)
