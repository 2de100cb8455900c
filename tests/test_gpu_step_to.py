"""sldg_step_to: the out-of-place Strang step (include/sldg.h) against sldg_step -- same 1-D sweeps in the same
order, so f, rho and E must agree BIT FOR BIT -- on ping-pong sequences between two caller buffers and between the caller's
buffer and the workspace buffer (sldg_workspace_field); the end-of-step field option; argument errors."""
import ctypes as C

import numpy as np
import pytest
import torch

import workloads as W

pytestmark = pytest.mark.gpu

# (index into W.CONFIGS, cells): every dim_x / dim_v combination of the BASELINE configs at sizes that reach the fused passes
CASES = [(0, [8, 8, 16, 16]), (1, [12, 10, 12, 10]), (2, [10, 8, 8, 6, 6]), (3, [6, 4, 4, 8, 6, 5]), (4, [4, 6, 4, 20, 5, 4])]


@pytest.fixture(scope="module")
def P():
    import paper_2110_14557_b200 as pkg
    if not torch.cuda.is_available():
        pytest.fail("gpu test without a CUDA device")
    return pkg


def fresh(P, cfg, prec="f64"):
    g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], precision=prec)
    f = W.initial_data(cfg, [g.node_coords(a) for a in range(g.d)]).to(g.dtype).to(g.device).contiguous()
    return g, f


@pytest.mark.parametrize("case", CASES, ids=lambda c: f"{W.CONFIGS[c[0]]['name']}-{'x'.join(map(str, c[1]))}")
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_step_to_equals_step_bit_for_bit(P, case, prec):
    cfg = W.scaled(W.CONFIGS[case[0]], case[1])
    dt = cfg["dt"]
    g, f = fresh(P, cfg, prec)
    g.set_option("graph", 0)
    ref = f.clone()
    a, b = f.clone(), torch.full_like(f, float("nan"))
    n0 = g.launch_count()
    for s in range(3):
        g.step(ref, dt)
        rho_ref, E_ref = g.last_rho(), g.last_E()
        g.step_to(a, b, dt)
        assert torch.equal(b, ref), (s, int((b != ref).sum()))
        assert torch.equal(g.last_rho(), rho_ref) and torch.equal(g.last_E(), E_ref)
        a, b = b, a
    # ping-pong between the caller's buffer and the workspace buffer: no third |f|-sized array
    w = g.workspace_field()
    assert w.shape == f.shape and w.data_ptr() != f.data_ptr()
    cur, oth = f, w
    for s in range(4):
        g.step_to(cur, oth, dt)
        cur, oth = oth, cur
    for s in range(1):
        g.step(ref, dt)
    assert torch.equal(cur, ref)
    assert cur.data_ptr() == f.data_ptr()                       # an even number of calls ends in the caller's buffer


def test_step_to_end_of_step_field_is_the_field_of_the_new_state(P):
    cfg = W.scaled(W.CONFIGS[3], [6, 4, 4, 8, 6, 5])
    g, f = fresh(P, cfg)
    out = torch.empty_like(f)
    g.step_to(f.clone(), out, cfg["dt"], end_of_step_field=True)
    rho = g.density(out)
    E = g.poisson(rho)
    assert torch.equal(g.last_rho(), rho) and torch.equal(g.last_E(), E)
    out2 = torch.empty_like(f)
    g.step_to(f.clone(), out2, cfg["dt"])
    assert torch.equal(out, out2) and not torch.equal(g.last_rho(), rho)      # without the option: rho of the half step


def test_step_to_uses_fewer_passes_than_step(P):
    cfg = W.scaled(W.CONFIGS[3], [6, 4, 4, 8, 6, 5])
    g, f = fresh(P, cfg)
    g.set_option("graph", 0); g.set_option("fuse_v3", 2)
    g.timing_enable(True); g.timing_read()
    g.step_to(f, torch.empty_like(f), cfg["dt"])
    kinds, _ = g.timing_read()
    g.timing_enable(False)
    sweeps = sum(v[0] for name, v in kinds.items() if name.startswith("sweep"))
    want = P.plan_query_step_to(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], fuse_v3=2)
    assert sweeps == want["x_passes"] + want["v_passes"] == 3 and kinds["copies"][0] == 0 and kinds["rho"][0] == 1


def test_step_to_rejects_bad_arguments(P):
    cfg = W.scaled(W.CONFIGS[0], [4, 4, 4, 4])
    g, f = fresh(P, cfg)
    L = P.lib()
    p = C.c_void_p(f.data_ptr())
    assert L.sldg_step_to(g._h, p, p, 0.1, 0) == -1              # in place
    assert L.sldg_step_to(g._h, None, p, 0.1, 0) == -1
    assert L.sldg_step_to(g._h, p, None, 0.1, 0) == -1
    assert L.sldg_step_to(g._h, p, C.c_void_p(f.data_ptr() + 8), 0.1, 0) == -1   # misaligned
    assert L.sldg_workspace_field(None) is None
