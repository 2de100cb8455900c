"""GPU parity of the single precision mode (sldg_create_prec(..., SLDG_F32), SURVEY 8(f) rank 2,
reading W) against the oracle's fp32 functions on the same seeded float32 inputs.

Bars.  The two sides round A, B to fp32 from fp64 values that agree to 1e-15, then the GPU uses fused multiply-add
chains where the oracle rounds every product and sum: per sweep the difference is at most (2(k+1)+1) ulp32 of
sum|A||u| <= about 1e-6 max|u|; bar 2e-6 per sweep, 2e-5 after 10 Strang steps.  Integer shifts: bit-exact.
rho and E are fp64 on both sides: compared relative to their own size at the accumulated fp32 error of f.
"""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import oracle as O

pytestmark = pytest.mark.gpu

TOL_SWEEP = 2e-6
TOL_STEPS = 2e-5


def rel_inf(g, o):
    return float(np.abs(g.astype(np.float64) - o.astype(np.float64)).max() / np.abs(o).max())


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
    return (P.Sldg(dx, dv, cells, k, dom, precision="f32"),
            O.Oracle(dx, dv, cells, k, dom, threads=O.lib().orc_max_threads()))


GEOMS = [
    (1, 1, [37, 23], 1),
    (1, 2, [16, 5, 7], 2),
    (2, 2, [8, 8, 16, 16], 1),        # BASELINE config 1
    (2, 2, [7, 5, 6, 9], 2),          # odd D everywhere: scalar / non-TMA paths
    (2, 2, [5, 3, 4, 3], 0),
    (2, 2, [6, 4, 5, 3], 3),
    (2, 2, [4, 3, 3, 2], 4),
    (2, 3, [6, 4, 5, 4, 3], 1),
    (3, 3, [4, 3, 5, 3, 4, 2], 1),
    (2, 2, [40, 33, 6, 5], 1),
    (2, 2, [64, 9, 3, 4], 2),
]
KINDS_FRAC = ["small", "cfl", "edge"]
KINDS_INT = ["int0", "int+1", "int-3", "intwrap", "intmix"]


@pytest.mark.parametrize("geom", GEOMS, ids=lambda g: f"{g[0]}x{g[1]}v-{'x'.join(map(str, g[2]))}-k{g[3]}")
def test_every_axis_every_shift_kind_f32(P, geom):
    dx, dv, cells, k = geom
    g, o = make_pair(P, dx, dv, cells, k)
    f0 = W.random_field(o.shape, seed=W.SEED + k).to(torch.float32)
    f0.view(-1)[::11] = -0.0
    for axis in range(dx + dv):
        n = o.D[dx + axis] if axis < dx else o.X
        for kind in KINDS_FRAC + KINDS_INT:
            delta = W.delta_table(n, kind, seed=W.SEED + axis, ncells=cells[axis]).numpy()
            want = o.sweep_axis_f32(f0.numpy(), axis, delta)
            fg = f0.to(g.device).contiguous()
            g.advect_axis(fg, axis, delta)
            got = fg.cpu().numpy()
            assert got.dtype == np.float32
            if kind in KINDS_INT:
                assert np.array_equal(got.view(np.int32), want.view(np.int32)), (axis, kind)
            else:
                assert rel_inf(got, want) <= TOL_SWEEP, (axis, kind, rel_inf(got, want))


def small_cfgs():
    c = W.CONFIGS
    return [c[0], W.scaled(c[1], [12, 10, 8, 8]), W.scaled(c[2], [8, 8, 6, 6, 4]), W.scaled(c[3], [6, 4, 4, 6, 4, 4]),
            W.scaled(c[4], [6, 4, 6, 4, 6, 4]), W.NEXT_CONFIGS[0]]


@pytest.mark.parametrize("cfg", small_cfgs(), ids=lambda c: c["name"])
def test_parts_and_ten_strang_steps_f32(P, cfg):
    g, o = make_pair(P, cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
    f0 = W.initial_data(cfg, [o.node_coords(a) for a in range(o.d)]).to(torch.float32)
    dt = cfg["dt"]
    # advect_x (fused and unfused plans agree bit for bit), density, advect_v
    outs = []
    for fuse, xcopy in ((1, 1), (0, 0), (1, 0)):
        g.set_option("fuse_x", fuse); g.set_option("x_copy", xcopy)
        fg = f0.to(g.device).contiguous()
        g.advect_x(fg, dt / 2)
        outs.append(fg.cpu().numpy())
    g.set_option("fuse_x", 1); g.set_option("x_copy", 0)
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
    want = o.advect_x_f32(f0.numpy(), dt / 2)
    assert rel_inf(outs[0], want) <= TOL_SWEEP * cfg["dim_x"]
    rho_g = g.density(fg).cpu().numpy()
    assert np.abs(rho_g - o.density_f32(outs[0])).max() <= 1e-13 * np.abs(rho_g).max()
    E = o.poisson(o.density_f32(want))
    Ed = torch.from_numpy(E).to(g.device)
    g.advect_v(fg, Ed, dt)
    assert rel_inf(fg.cpu().numpy(), o.advect_v_f32(outs[0], E, dt)) <= TOL_SWEEP * cfg["dim_x"]
    # 10 Strang steps
    fg, fo = f0.to(g.device).contiguous(), f0.numpy()
    m0 = g.mass(fg)
    for _ in range(10):
        g.step(fg, dt)
        fo, rho_o, E_o = o.step_f32(fo, dt)
    assert fg.dtype == torch.float32
    assert rel_inf(fg.cpu().numpy(), fo) <= TOL_STEPS
    assert np.abs(g.last_rho().cpu().numpy() - rho_o).max() <= TOL_STEPS * np.abs(rho_o).max()
    assert np.abs(g.last_E().cpu().numpy() - E_o).max() <= TOL_STEPS * max(1.0, np.abs(E_o).max())
    assert abs(g.mass(fg) - m0) <= 5e-6 * abs(m0)
    assert abs(g.mass(fg) - o.mass_f32(fg.cpu().numpy())) <= 1e-12 * abs(m0)


def test_f32_and_f64_contexts_reject_the_wrong_buffers(P):
    g = P.Sldg(1, 1, [4, 4], 1, [0, 1, -1, 1], precision="f32")
    assert P.lib().sldg_precision(g._h) == 1
    with pytest.raises(AssertionError):
        g.advect_x(torch.zeros(g.shape, dtype=torch.float64, device=g.device), 0.1)
    assert g.workspace.numel() < P.Sldg(1, 1, [4, 4], 1, [0, 1, -1, 1]).workspace.numel()
