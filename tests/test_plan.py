"""Host logic (no GPU): the pass budget of the step plans, through sldg_plan_query.

sldg_plan_query runs the library's own planning code (x_plan / step_best / sldg_steps, buffer-flip parities included)
with every launch replaced by a counter, so these numbers are those of the real calls with option graph = 0 (the
CUDA-graph replay of small problems is not modelled).  What is checked: P:66-72 -- a Strang step is x(dt/2), field
solve, v(dt), x(dt/2); P:199 -- every advection reads and writes f once; DESIGN.md section 6 -- which sweeps share a
pass.  A plan must always end in the caller's buffer WITHOUT a device copy.
"""
import itertools

import pytest

import paper_2110_14557_b200 as P
import workloads as W


def q(cfg, n, **kw):
    return P.plan_query(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], n, **kw)


CFG = {c["name"].split("_")[0]: c for c in W.CONFIGS}


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5"])
def test_single_step_budget(name):
    """One sldg_step must end in f: two one-pass x half steps and two v passes (dim_x = 2: the two walks, the fused
    v_1+v_2 pass would cost a two-pass x half step; dim_x = 3: the fused pass plus the v_3 walk)."""
    r = q(CFG[name], 0)
    assert (r["x_passes"], r["v_passes"], r["rho_passes"], r["field_solves"], r["copies"]) == (2, 2, 1, 1, 0)


@pytest.mark.parametrize("name,x,v", [("cfg2", 11, 11), ("cfg3", 11, 11), ("cfg4", 20, 10), ("cfg5", 20, 10)])
def test_ten_steps_budget(name, x, v):
    """sldg_steps(10).  dim_x = 2: first half step 1 pass, 9 merged double half steps, 9 fused v passes and the last v
    advection as two walks (so that the flips before the closing half step are odd and it is ONE pass).  dim_x = 3: 2 x
    passes and ONE v pass (v_1+v_2+v_3 fused) per step."""
    r = q(CFG[name], 10)
    assert (r["x_passes"], r["v_passes"], r["rho_passes"], r["field_solves"], r["copies"]) == (x, v, 10, 10, 0)


def test_options_change_the_budget_as_documented():
    c2, c4 = CFG["cfg2"], CFG["cfg4"]
    assert q(c2, 10, x_double=0)["x_passes"] == 20 and q(c2, 10, x_double=0)["v_passes"] == 10     # alternating buffers
    r = q(c2, 10, x_double=0, fuse_v=0)
    assert (r["x_passes"], r["v_passes"]) == (20, 20)
    r = q(c4, 10, fuse_v=0, fuse_v3=0)           # three v walks: odd flips, sldg_steps alternates buffers
    assert (r["x_passes"], r["v_passes"]) == (20, 30)
    r = q(c4, 10, fuse_v3=0)                     # fused v_1+v_2 + the v_3 walk
    assert (r["x_passes"], r["v_passes"]) == (20, 20)
    r = q(c4, 0, fuse_v=0, fuse_v3=0)            # a single step: one x half step needs two passes
    assert (r["x_passes"], r["v_passes"]) == (3, 3)
    r = q(c4, 0, fuse_v=0)                       # a single step with the one-pass v advection only: the odd flip costs an x pass
    assert (r["x_passes"], r["v_passes"]) == (3, 1)
    r = q(c4, 10, x_double=2)                    # forced double x_1x_2x_3 pass (slower than two passes on B200: not the default)
    assert (r["x_passes"], r["v_passes"], r["copies"]) == (11, 11, 0)
    r = q(c2, 0, fuse_v=2)                       # forced fused v in a single dim_x = 2 step: the odd flip costs an x pass
    assert (r["x_passes"], r["v_passes"]) == (3, 1)
    r = q(c2, 10, precision="f32")               # single precision: no automatic fused v for dim_x = 2
    assert (r["x_passes"], r["v_passes"]) == (12, 20)
    r = q(c2, 2)                                 # two steps: one merged pass, the last v as walks, one-pass closing half step
    assert (r["x_passes"], r["v_passes"], r["copies"]) == (3, 3, 0)


def test_degree_three_fuses_v_but_not_the_x_half_steps():
    """k = 3 (the paper's default order): the fused v pass exists (256-thread blocks), the double x half step
    does not (two walk states of (k+1)^2 values do not fit the register file) -> sldg_steps alternates buffers."""
    cfg = {c["name"]: c for c in W.NEXT_CONFIGS}["bot_5d_k3_16"]
    r = q(cfg, 10)
    assert (r["x_passes"], r["v_passes"], r["copies"]) == (20, 10, 0)
    r = q(cfg, 10, fuse_v=0)
    assert (r["x_passes"], r["v_passes"], r["copies"]) == (20, 20, 0)


@pytest.mark.parametrize("dx,dv", [(1, 1), (1, 2), (2, 2), (2, 3), (3, 3)])
@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_every_plan_ends_in_the_callers_buffer_without_a_copy(dx, dv, k):
    cells = [6, 5, 4, 6, 5, 4][:dx + dv]
    big = [64, 48, 40, 24, 20, 16][:dx + dv]
    for cc, n, safe, fv, xd, prec, fv3 in itertools.product((cells, big), (0, 1, 2, 3, 4, 7), (True, False), (0, 1, 2), (0, 1, 2) if dx == 3 else (0, 1),
                                                            ("f64", "f32"), (0, 1, 2) if dx == 3 else (1,)):
        r = P.plan_query(dx, dv, cc, k, n, precision=prec, shifts_below_one=safe, fuse_v=fv, x_double=xd, fuse_v3=fv3)
        steps = max(1, n)
        assert r["copies"] == 0, (cc, n, safe, fv, xd, prec, fv3, r)
        assert r["rho_passes"] == steps and r["field_solves"] == steps
        # never more passes than one per 1-D sweep, never fewer than the merged minimum
        assert r["x_passes"] <= 2 * dx * steps and r["v_passes"] <= dx * steps
        assert r["x_passes"] >= steps + 1 and r["v_passes"] >= steps


def test_out_of_place_step_has_the_pass_budget_of_merged_steps():
    """sldg_step_to (result in the other buffer) may flip the buffers an odd number of times: one step of the 3x3v
    configs is 3 passes + rho (sldg_step: 4), of the dim_x = 2 configs 3 passes (sldg_step: 4); the end-of-step field evaluation
    of PAPER.md:199 adds exactly one rho pass and one field solve; never a whole-array copy."""
    import paper_2110_14557_b200 as P
    for dx, dv, cells, k in [(3, 3, [24, 24, 24, 20, 20, 20], 1), (3, 3, [20] * 6, 1), (2, 2, [64] * 4, 2), (2, 3, [32] * 5, 1)]:
        one = P.plan_query(dx, dv, cells, k, 0)
        to = P.plan_query_step_to(dx, dv, cells, k)
        diag = P.plan_query_step_to(dx, dv, cells, k, end_of_step_field=True)
        assert one["x_passes"] + one["v_passes"] == 4
        assert (to["x_passes"], to["v_passes"], to["rho_passes"], to["field_solves"], to["copies"]) == (2, 1, 1, 1, 0)
        assert (diag["x_passes"], diag["v_passes"], diag["rho_passes"], diag["field_solves"], diag["copies"]) == (2, 1, 2, 2, 0)
    # degree 3 (no one-pass 3x3v sweeps yet): no worse than sldg_step
    one, to = P.plan_query(3, 3, [9] * 6, 3, 0), P.plan_query_step_to(3, 3, [9] * 6, 3)
    assert to["x_passes"] + to["v_passes"] <= one["x_passes"] + one["v_passes"] and to["copies"] == 0
