"""CPU checks (world_size 2, gloo) of the v-axis domain decomposition plumbing (paper_2110_14557_b200/shard.py;
PAPER.md:129-131, Fig. 3; SURVEY 8(f) rank 4 tail): slab geometry, halo width, halo exchange on a periodic ring, the rho
all-reduce and the redundant field solve.  The arithmetic is supplied by an engine; here the engine is the CPU oracle on
CPU buffers (test infrastructure), on a GPU it is the CUDA context -- the plumbing under test is the same.  The sharded
steps must reproduce the single-domain oracle steps on every rank's interior (up to the summation order of rho).
"""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np
import torch
import torch.distributed as dist
import workloads as W
from oracle import oracle as O
from paper_2110_14557_b200 import shard as S

case = json.loads({case!r})
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
if world > 1:
    dist.init_process_group(backend="gloo")

class OracleEngine:
    # the CPU oracle behind the engine interface of shard.VShard (arrays are CPU torch tensors, updated in place)
    def __init__(self, g):
        self.o = O.Oracle(g.dim_x, g.dim_v, g.cells, g.degree, g.domain, threads=2)
    def advect_x(self, f, tau):
        f.copy_(torch.from_numpy(self.o.advect_x(f.numpy(), tau)))
    def advect_v(self, f, E, tau):
        f.copy_(torch.from_numpy(self.o.advect_v(f.numpy(), E.numpy(), tau)))
    def density(self, f):
        return torch.from_numpy(self.o.density(np.ascontiguousarray(f.numpy())))
    def poisson(self, rho):
        return torch.from_numpy(self.o.poisson(rho.numpy()))

cfg = W.scaled(W.CONFIGS[case["config"]], case["cells"])
geom = S.Geometry(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"])
dt, nsteps = case["dt"], case["nsteps"]
# the full problem (every rank computes it: the reference of the comparison)
full = O.Oracle(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], threads=2)
f_full = W.initial_data(cfg, [full.node_coords(a) for a in range(full.d)]).numpy() * case["scale"]
ref, emax = f_full, 0.0
for _ in range(nsteps):
    ref, rho_ref, E_ref = full.step(ref, dt)
    emax = max(emax, float(np.abs(E_ref[-1]).max()))
H = S.halo_cells(geom, 1.05 * emax, dt)
sh = S.VShard(geom, rank, world, H, OracleEngine, dist if world > 1 else None)
# this rank's extended slab of the initial data (halo cells start as garbage: the first exchange fills them)
k1 = cfg["degree"] + 1
r0 = sh.start * k1
f_ext = torch.full(tuple(reversed([c * k1 for c in sh.extended.cells])), float("nan"), dtype=torch.float64)
sh.interior_of(f_ext).copy_(torch.from_numpy(f_full[r0:r0 + sh.n_loc * k1]))
if H:
    f_ext[:H * k1] = 0.0; f_ext[f_ext.shape[0] - H * k1:] = 0.0      # finite garbage (x sweeps touch the halos too)
for _ in range(nsteps):
    rho, E = sh.step(f_ext, dt)
got = sh.interior_of(f_ext).numpy()
want = ref[r0:r0 + sh.n_loc * k1]
err = float(np.abs(got - want).max() / np.abs(ref).max())
err_rho = float(np.abs(rho.numpy() - rho_ref).max() / np.abs(rho_ref).max())
err_E = float(np.abs(E.numpy() - E_ref).max() / max(np.abs(E_ref).max(), 1e-300))
if world > 1:
    dist.barrier(); dist.destroy_process_group()
print(json.dumps(dict(rank=rank, H=H, n_loc=sh.n_loc, err=err, err_rho=err_rho, err_E=err_E, finite=bool(np.isfinite(got).all()))))
"""

CASES = [
    # 2x2v: the cut axis v_2 is advected; a strong field so that the halo is several cells wide
    dict(config=0, cells=[4, 4, 6, 12], dt=0.5, nsteps=2, scale=40.0),
    dict(config=0, cells=[4, 4, 6, 8], dt=0.1, nsteps=3, scale=1.0),
    # 2x3v: the cut axis v_3 is not advected (reading D): no halo
    dict(config=2, cells=[4, 4, 4, 4, 6], dt=0.1, nsteps=2, scale=1.0),
    # 3x3v: v_3 advected and cut
    dict(config=3, cells=[3, 2, 2, 3, 2, 6], dt=0.2, nsteps=2, scale=20.0),
]


def run_ranks(tmp_path, case, world, port):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, case=json.dumps(case)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), CUDA_VISIBLE_DEVICES="",
               OMP_NUM_THREADS="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(world)]
    outs = [p.communicate(timeout=300) for p in procs]
    res = []
    for p, (so, se) in zip(procs, outs):
        assert p.returncode == 0, se[-3000:]
        res.append(json.loads(so.strip().splitlines()[-1]))
    return res


@pytest.mark.parametrize("ci", range(len(CASES)))
def test_two_rank_sharded_steps_equal_the_single_domain_steps(tmp_path, ci):
    case = CASES[ci]
    res = run_ranks(tmp_path, case, 2, 29641 + ci)
    for d in res:
        assert d["finite"] and d["err"] <= 1e-13 and d["err_rho"] <= 1e-13 and d["err_E"] <= 1e-11, d
    if ci == 0:
        assert res[0]["H"] >= 3                               # the strong-field case really needs a wide halo
    if ci == 2:
        assert res[0]["H"] == 0                               # 2x3v: nothing to exchange


def test_three_ranks_with_uneven_slabs(tmp_path):
    """8 cells of the cut axis over 3 ranks: slabs of 3, 3 and 2 cells (the 20 v_3 cells of cfg4 / cfg5 do not divide by 8 either)."""
    res = run_ranks(tmp_path, CASES[1], 3, 29661)
    assert sorted(d["n_loc"] for d in res) == [2, 3, 3]
    for d in res:
        assert d["finite"] and d["err"] <= 1e-13 and d["err_rho"] <= 1e-13 and d["err_E"] <= 1e-11, d


def test_slab_bounds_of_uneven_cuts():
    sys.path.insert(0, ROOT)
    from paper_2110_14557_b200 import shard as S

    class Nothing:
        def __init__(self, g): self.g = g
    geom = S.Geometry(3, 3, [2, 2, 2, 2, 2, 20], 1, [0, 1] * 5 + [-6, 6])
    sl = [S.VShard(geom, r, 8, 2, Nothing) for r in range(8)]
    assert [s.n_loc for s in sl] == [3, 3, 3, 3, 2, 2, 2, 2] and [s.start for s in sl] == [0, 3, 6, 9, 12, 14, 16, 18]
    for a, b in zip(sl, sl[1:]):
        assert a.interior.domain[-1] == pytest.approx(b.interior.domain[-2], abs=1e-15)
    assert sl[0].interior.domain[-2] == -6 and sl[-1].interior.domain[-1] == pytest.approx(6)
    assert sl[4].extended.cells[-1] == 2 + 4
    with pytest.raises(ValueError):
        S.VShard(geom, 0, 8, 3, Nothing)                      # halo wider than the smallest slab


def test_single_rank_shard_is_the_periodic_problem(tmp_path):
    """world = 1: the halo exchange degenerates to the periodic wrap of the rank's own slab."""
    res = run_ranks(tmp_path, CASES[1], 1, 29651)
    assert res[0]["err"] <= 1e-13 and res[0]["n_loc"] == CASES[1]["cells"][-1]


def test_halo_width_rule():
    sys.path.insert(0, ROOT)
    from paper_2110_14557_b200 import shard as S
    g = S.Geometry(2, 2, [4, 4, 6, 8], 1, [0, 1, 0, 1, -6, 6, -6, 6])     # h_v = 1.5 on the cut axis
    assert S.halo_cells(g, 0.0, 0.1) == 1                                 # donors i and i-1
    assert S.halo_cells(g, 15.0, 0.1) == 2                                # |delta| = 1 cell
    assert S.halo_cells(g, 31.0, 0.1) == 4                                # |delta| = 2.07 cells
    g3 = S.Geometry(2, 3, [4, 4, 4, 4, 6], 1, [0, 1] * 2 + [-6, 6] * 3)
    assert S.halo_cells(g3, 100.0, 0.1) == 0                              # cut axis not advected
    assert S.VShard(g, 0, 3, 1, lambda geom: None).n_loc == 3             # 8 cells over 3 ranks: uneven slabs (3, 3, 2) are allowed
    with pytest.raises(ValueError):
        S.VShard(g, 0, 9, 1, lambda geom: None)                           # more ranks than cells


def test_step_refuses_a_field_that_outgrew_the_halo():
    """VShard.step checks max|E| on the cut axis against the halo width it was built with (advisor finding, round 2): a field
    that has grown past the construction-time estimate must raise, not wrap silently."""
    import torch
    from paper_2110_14557_b200 import shard as S

    class FakeEngine:                       # plumbing only: a field of a chosen size, no arithmetic
        emax = 0.5
        def __init__(self, g):
            self.g = g
        def advect_x(self, f, tau): pass
        def advect_v(self, f, E, tau): pass
        def density(self, f): return torch.zeros(4)
        def poisson(self, rho): return torch.full((2, 4), FakeEngine.emax, dtype=torch.float64)

    geom = S.Geometry(2, 2, [2, 2, 8, 8], 1, [0, 1, 0, 1, -4, 4, -4, 4])          # h_v = 1
    dt = 1.0
    H = S.halo_cells(geom, 0.5, dt)                                               # ceil(0.5) + 1 = 2
    assert H == 2
    sh = S.VShard(geom, 0, 1, H, FakeEngine)
    f_ext = torch.zeros(tuple(reversed([c * 2 for c in sh.extended.cells])), dtype=torch.float64)
    sh.step(f_ext, dt)                                                            # |delta| = 0.5 <= H - 1: fine
    FakeEngine.emax = 1.0
    sh.step(f_ext, dt)                                                            # |delta| = 1.0 = H - 1: still fine
    FakeEngine.emax = 1.25
    with pytest.raises(S.HaloTooNarrow):
        sh.step(f_ext, dt)                                                        # needs 3 cells
    # the interior-density hook replaces the second engine
    calls = []
    sh2 = S.VShard(geom, 0, 1, H, FakeEngine, interior_density=lambda fi: calls.append(tuple(fi.shape)) or torch.zeros(4))
    assert sh2.eng_int is None
    FakeEngine.emax = 0.5
    sh2.step(f_ext, dt)
    assert calls == [tuple(sh2.interior_of(f_ext).shape)]
