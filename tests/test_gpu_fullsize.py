"""GPU parity at BASELINE.json's FULL sizes (configs 2-5), in the launch configuration bench.py times.

The oracle cannot hold 10-57 GB arrays, but every operation of the path decouples: x-sweeps act on x-space for a
fixed velocity node, v-sweeps and the density on v-space for a fixed x node.  So the test gathers, from the
full-size device array, the complete x-space of a few velocity CELLS and the complete v-space of a few x CELLS,
runs the full-size GPU call, and compares those slabs with the oracle applied to the same slabs as a small problem
(one cell per frozen axis).  Poisson runs on the full-size rho directly.  Single sweeps with random shift tables
(CFL > 1 and integer) are checked on sampled lines with the oracle's line routine.
Bars as in test_gpu_parity.py: 1e-12 per sweep, bit-exact for integer shifts.
"""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import oracle as O

pytestmark = pytest.mark.gpu

TOL = 1e-12


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


@pytest.fixture(scope="module", params=[1, 2, 3, 4], ids=lambda i: W.CONFIGS[i]["name"])
def full(request, P):
    cfg = W.CONFIGS[request.param]
    need = 2 * W.field_elems(cfg) * 8 + (6 << 30)
    free, _ = torch.cuda.mem_get_info()
    if free < need:
        pytest.fail(f"{cfg['name']}: needs {need >> 30} GiB of device memory, {free >> 30} GiB free")
    g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
    f = g.empty_field()
    W.initial_data(cfg, [g.node_coords(a) for a in range(g.d)], device=g.device, out=f)
    W.perturb_inplace(f, seed=W.SEED + request.param)
    yield cfg, g, f
    g.close()
    del f
    torch.cuda.empty_cache()


@pytest.mark.parametrize("xcopy", [0, 1], ids=["even-parity plan", "odd-parity plan (the one-pass fused sweeps)"])
def test_advect_x_on_full_x_space_of_sampled_velocity_cells(full, xcopy):
    """x_copy = 1 runs the plan sldg_step / sldg_steps use for their flipping x half steps: the fused x1+x2 pass
    (dim_x = 2) or the fused x1+x2+x3 pass (dim_x = 3), in the launch configuration bench.py times."""
    cfg, g, f = full
    g.set_option("x_copy", xcopy)
    dx, dv = cfg["dim_x"], cfg["dim_v"]
    vaxes = list(range(dx, dx + dv))
    cells = cell_samples(cfg["cells"][dx:], 5, seed=1)
    before = [f[slab_index(g, vaxes, c)].cpu().numpy() for c in cells]
    tau = cfg["dt"] / 2
    m0 = g.mass(f)
    g.advect_x(f, tau)
    assert abs(g.mass(f) - m0) <= 1e-12 * abs(m0)
    for c, b in zip(cells, before):
        dom = list(cfg["domain"][:2 * dx])
        for a, i in zip(vaxes, c):
            dom += cell_domain(cfg, a, i)
        o = O.Oracle(dx, dv, cfg["cells"][:dx] + [1] * dv, cfg["degree"], dom, threads=O.lib().orc_max_threads())
        want = o.advect_x(b, tau)
        got = f[slab_index(g, vaxes, c)].cpu().numpy()
        assert rel_inf(got, want) <= TOL * dx, (c, rel_inf(got, want))
    g.set_option("x_copy", 0)


def test_density_poisson_advect_v_on_full_v_space_of_sampled_x_cells(full):
    cfg, g, f = full
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
    for o, b, sl in zip(smalls, before, xsl):
        assert np.abs(rho_h[sl] - o.density(b)).max() <= TOL * scale
    # Poisson on the full-size rho (the oracle's naive DFT handles X <= 110592)
    ofull = O.Oracle(dx, dv, cfg["cells"][:dx] + [1] * dv, cfg["degree"],
                     list(cfg["domain"][:2 * dx]) + [0.0, 1.0] * dv, threads=O.lib().orc_max_threads())
    E = g.poisson(rho)
    E_h = E.cpu().numpy()
    E_o = ofull.poisson(rho_h)
    assert rel_inf(E_h, E_o) <= 1e-11, rel_inf(E_h, E_o)
    # advect_v with the physical field and with a strong seeded field (|delta| up to ~3 cells)
    hv = (cfg["domain"][2 * dx + 1] - cfg["domain"][2 * dx]) / cfg["cells"][dx]
    dt = cfg["dt"]
    strong = W.random_E(dx, g.xshape, amplitude=3.0 * hv / dt, device=g.device)
    for Efield in (E, strong):
        Eh = Efield.cpu().numpy()
        m0 = g.mass(f)
        g.advect_v(f, Efield, dt)
        assert abs(g.mass(f) - m0) <= 1e-12 * abs(m0)
        after = []
        for o, b, c, sl in zip(smalls, before, cells, xsl):
            want = o.advect_v(b, np.ascontiguousarray(Eh[(slice(None),) + sl]), dt)
            got = f[slab_index(g, xaxes, c)].cpu().numpy()
            assert rel_inf(got, want) <= TOL * dx, (c, rel_inf(got, want))
            after.append(got)
        before = after


@pytest.mark.parametrize("kind", ["cfl", "intmix"])
def test_single_sweeps_on_sampled_lines(full, kind):
    """Every swept axis through the test hook at full size; 4096 seeded lines per axis against orc_sweep_line."""
    cfg, g, f = full
    dx = cfg["dim_x"]
    k = cfg["degree"]
    rng = np.random.default_rng(7)
    for axis in range(2 * dx):
        Da = g.D[axis]
        inner = int(np.prod(g.D[:axis], dtype=np.int64)) if axis else 1
        outer = g.nf // (inner * Da)
        n = g.D[dx + axis] if axis < dx else g.X
        delta = W.delta_table(n, kind, seed=W.SEED + axis, ncells=cfg["cells"][axis]).numpy()
        ns = 4096
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
        want = np.stack([O.sweep_line(k, lines_in[i], delta[sidx[i]]) for i in range(ns)])
        if kind == "intmix":
            assert np.array_equal(lines_out, want), axis
        else:
            assert rel_inf(lines_out, want) <= TOL, (axis, rel_inf(lines_out, want))


def test_constants_are_preserved_by_two_steps_at_full_size(full):
    """rows of A + B sum to 1 (invariant p4), so a constant f stays constant to round-off through
    every sweep of sldg_steps at full size (fused passes, in-place walks, v sweeps with E = 0 up to round-off).
    Runs last: it overwrites the module's f."""
    cfg, g, f = full
    f.fill_(0.375)
    g.steps(f, cfg["dt"], 2)
    lo, hi = float(f.min()), float(f.max())
    assert abs(lo - 0.375) <= 1e-13 and abs(hi - 0.375) <= 1e-13, (lo, hi)
