#!/usr/bin/env python
"""bench.py -- one JSON line for the driver.

    python bench.py --gpus N --steps K --warmup W [--impl reference] [--config I]

A "step" is one Strang step (3*d_x sweeps + rho + Poisson + shift tables) of the
SLDG Vlasov-Poisson path on synthetic data of BASELINE.json configs[I] (default I=4: cfg5, 6-d two-stream,
24^3 x 20^3 cells, k=1, 48^3*40^3 values = 56.6 GB fp64: the largest configuration that fits one B200; the
other four configs are run briefly in the same invocation and attached under `configs`).  Metric: effective
HBM GB/s per 1-D advection sweep, 2*|f|*8 B per sweep / time (BASELINE.json `metric`); `value` uses the WHOLE
step time (rho, Poisson and table kernels included).  Because fused / merged passes perform several sweeps per
trip over f, the line also carries the PHYSICAL traffic (`physical_bytes_per_step`, `physical_frac`, and per
launch kind under `kernels`): passes * 2*|f|*8 B + the rho read, over the measured copy rate.  Multi-GPU: the path does not shard in this build ("replicas only"): every rank
runs an independent replica, value = total bytes of all ranks / max-over-ranks time.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "effective HBM GB/s per 1D advection sweep (2*|f|*8 B / time), whole Strang step"
UNIT = "GB/s"
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json north_star "~8 TB/s"
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy burst)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def sweeps_per_step(cfg):
    return 3 * cfg["dim_x"]


ESIZE = 8                         # bytes per value of f; --dtype f32 (single precision mode) sets 4


def sweep_bytes(cfg):
    import workloads as W
    return 2 * W.field_elems(cfg) * ESIZE


# ----------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._halt = index, [], threading.Event()

    def run(self):
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
                if out.returncode == 0 and out.stdout.strip():
                    self.rows.append([c.strip() for c in out.stdout.strip().split(",")])
            except Exception:
                pass
            self._halt.wait(0.1)

    def stop(self):
        self._halt.set()
        self.join(timeout=10)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows for n, v in zip(names, r[3:7]) if v.lower().startswith("active")})
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# ----------------------------------------------------------------------------- distributed plumbing
def dist_setup(n_gpus):
    """-> (rank, world, local_rank).  Under torchrun: init the process group (nccl on GPU, gloo otherwise)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        if torch.cuda.is_available():
            torch.cuda.set_device(local)
        dist.init_process_group(backend=backend)
    return rank, world, local


def aggregate(ms_local, bytes_local, device="cpu"):
    """Replicas-only aggregation: (max over ranks of the timed region [ms], sum over ranks of the bytes).
    Works with gloo (CPU tests) and nccl."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), float(bytes_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    b = torch.tensor([float(bytes_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(b, op=dist.ReduceOp.SUM)
    return float(t.item()), float(b.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


# ----------------------------------------------------------------------------- the oracle as CPU baseline
def oracle_sample_cfg(cfg, target_values=2.0e7):
    """A bounded sample of the workload: same dimensions, degree, domain, dt and initial data, fewer cells
    (a 'scaled replica'), sized so that one oracle Strang step takes seconds."""
    import workloads as W
    d = cfg["dim_x"] + cfg["dim_v"]
    k1 = cfg["degree"] + 1
    per_axis = max(2, int(round(target_values ** (1.0 / d) / k1)))
    cells = [min(c, per_axis) for c in cfg["cells"]]
    return W.scaled(cfg, cells)


def time_oracle(cfg, steps, warmup, budget_s=25.0, threads=None):
    """Time the oracle AS IT STANDS (oracle/sldg_oracle.c, all host threads) on a bounded sample.
    -> dict(value [GB/s effective per sweep], ms_per_step, cores, sample, steps)."""
    import workloads as W
    from oracle import oracle as O
    s = oracle_sample_cfg(cfg)
    cores = threads if threads else O.lib().orc_max_threads()
    o = O.Oracle(s["dim_x"], s["dim_v"], s["cells"], s["degree"], s["domain"], threads=cores)
    f = W.initial_data(s, [o.node_coords(a) for a in range(o.d)]).numpy()
    ostep = o.step
    if ESIZE == 4:                        # single precision mode: the oracle's fp32 functions
        f, ostep = f.astype("float32"), o.step_f32
    for _ in range(max(0, warmup)):
        f, _, _ = ostep(f, s["dt"])
    done, t0 = 0, time.perf_counter()
    while done < steps:
        f, _, _ = ostep(f, s["dt"])
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    ms = 1e3 * dt / done
    value = sweeps_per_step(s) * sweep_bytes(s) / (ms * 1e-3) / 1e9
    return {"value": value, "unit": UNIT, "ms_per_step": ms, "cores": cores, "kind": "oracle", "steps": done,
            "sample": f"scaled replica of {cfg['name']}: cells {s['cells']} ({W.field_elems(s)} values), "
                      f"{done} Strang step(s), {cores} host thread(s)"}


def run_reference(args, cfg, rank, world):
    """--impl reference: for this tier the reference arm IS the oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return None
    r = time_oracle(cfg, args.steps, args.warmup, budget_s=120.0)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": r["steps"], "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": cfg["name"], "note": "CPU oracle on a bounded sample; " + r["sample"]},
        "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    return line


# ----------------------------------------------------------------------------- the CUDA path
def ncu_traffic(cfg_name, kernel):
    """dram bytes per launch of `kernel` on workload `cfg_name` from the committed ncu capture (profiles/), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    try:
        with open(p) as fh:
            for ln in fh:
                if ln.startswith("{"):
                    d = json.loads(ln)
                    if d.get("workload") == cfg_name and d.get("kernel") == kernel:
                        return d
    except Exception:
        pass
    return None


def fill_initial(W, g, cfg, f, dtype, dev):
    coords = [g.node_coords(a) for a in range(g.d)]
    if dtype == "f32":                    # the generator works in fp64: fill slab by slab along the slowest axis
        D = f.shape[0]
        step = max(1, D // 8)
        for a in range(0, D, step):
            b = min(D, a + step)
            f[a:b].copy_(W.initial_data(cfg, coords[:-1] + [coords[-1][a:b]], device=dev))
    else:
        W.initial_data(cfg, coords, device=dev, out=f)


SWEEP_KINDS_PREFIX = "sweep"


def measure_config(args, cfg, dev, local, steps, warmup, headline):
    """One workload on this rank's GPU: K Strang steps through sldg_steps (timed with CUDA events on the library's stream),
    the same K steps as K sldg_step calls, and once more with events around every launch.
    -> (dict of figures, ms of the timed region, effective bytes of the timed region, solver, field) ."""
    import torch
    import workloads as W
    import paper_2110_14557_b200 as P

    g = P.Sldg(cfg["dim_x"], cfg["dim_v"], cfg["cells"], cfg["degree"], cfg["domain"], device=dev, precision=args.dtype)
    f = g.empty_field()
    fill_initial(W, g, cfg, f, args.dtype, dev)
    if args.poisson == "cg":
        g.set_poisson_solver(1, tol=1e-3)
    for kv in args.option or []:              # tuning knobs of sldg_set_option (speed only, never results): name=value
        name, val = kv.split("=")
        g.set_option(name, int(val))
    dt = cfg["dt"]
    nf = W.field_elems(cfg)
    nsweeps = sweeps_per_step(cfg)
    bytes_step = nsweeps * sweep_bytes(cfg)
    pass_bytes = 2 * nf * ESIZE               # one pass over f: every value read once and written once

    # warm-up through the SAME entry point as the timed region (sldg_steps plans merged passes that single sldg_step calls
    # never launch: their kernels would otherwise be loaded -- CUDA loads a kernel lazily at its first launch -- inside the
    # timed region), then one single step for the kernels only that path uses
    g.steps(f, dt, max(warmup, 3))
    g.step(f, dt)
    torch.cuda.synchronize(dev)
    # ---- timed region: K Strang steps, no instrumentation inside
    launches0 = g.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    if headline:
        barrier()
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    g.steps(f, dt, steps)                     # K Strang steps through the multi-step entry point (sldg_steps)
    e1.record(g.stream)
    torch.cuda.synchronize(dev)
    if headline:
        barrier()
    ms_total_local = e0.elapsed_time(e1)
    launches = g.launch_count() - launches0
    # ---- for comparison: the same K steps as K separate sldg_step calls (f at every integer time t_n is materialised in
    # the caller's buffer, as a per-step diagnostic would need; no merging of x half steps across steps)
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s0.record(g.stream)
    for _ in range(steps):
        g.step(f, dt)
    s1.record(g.stream)
    torch.cuda.synchronize(dev)
    ms_single_calls = s0.elapsed_time(s1) / steps
    # ---- and as K sldg_step_to calls ping-ponging between f and the workspace buffer: f(t_n) exists after every step too, at
    # the pass budget of the merged plan (no third |f|-sized buffer)
    wsf = g.workspace_field()
    cur, oth = f, wsf
    g.step_to(cur, oth, dt); cur, oth = oth, cur                # untimed: loads the kernels this plan uses
    s0.record(g.stream)
    for _ in range(steps):
        g.step_to(cur, oth, dt)
        cur, oth = oth, cur
    s1.record(g.stream)
    torch.cuda.synchronize(dev)
    ms_step_to = s0.elapsed_time(s1) / steps
    if cur is not f:
        f.copy_(cur)
    # ---- the same K steps again with CUDA events around every launch (on the library's stream): per-kernel figures
    g.timing_enable(True)
    g.steps(f, dt, steps)                     # untimed, same plan: with events on, small problems leave the graph path (kernels load here)
    g.timing_read()
    g.steps(f, dt, steps)
    kinds, axes = g.timing_read()
    g.timing_enable(False)
    clocks = sampler.stop()
    ms_step = ms_total_local / steps

    peak, peak_src = measured_peak()
    # PHYSICAL traffic: every sweep launch (single, fused or merged) is one pass over f = |f| values read + |f| written;
    # the rho launch reads f once.  This is what the HBM actually moves, and what the roofline fraction is taken of.
    passes = {k: v for k, v in kinds.items() if k.startswith(SWEEP_KINDS_PREFIX) and v[0]}
    n_pass = sum(n for n, _ in passes.values())
    n_rho = kinds.get("rho", (0, 0.0))[0]
    n_copy = kinds.get("copies", (0, 0.0))[0]     # whole-array device copies of f (fallback plans only): |f| read + |f| written each
    phys_step = ((n_pass + n_copy) * pass_bytes + n_rho * nf * ESIZE) / steps
    kernels = {}
    for k, (n, ms) in passes.items():
        gbs = pass_bytes / (ms / n * 1e-3) / 1e9
        kernels[k] = {"launches": n, "avg_ms": ms / n, "physical_gbs": gbs, "frac_of_measured_peak": gbs / peak,
                      "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS, "bytes_per_launch": pass_bytes}
    if n_rho:
        n, ms = kinds["rho"]
        gbs = nf * ESIZE / (ms / n * 1e-3) / 1e9
        kernels["rho"] = {"launches": n, "avg_ms": ms / n, "physical_gbs": gbs, "frac_of_measured_peak": gbs / peak,
                          "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS, "bytes_per_launch": nf * ESIZE}
    if n_copy:
        n, ms = kinds["copies"]
        gbs = pass_bytes / (ms / n * 1e-3) / 1e9
        kernels["copies"] = {"launches": n, "avg_ms": ms / n, "physical_gbs": gbs, "frac_of_measured_peak": gbs / peak,
                             "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS, "bytes_per_launch": pass_bytes}
    # EFFECTIVE per-axis figures (BASELINE.json's metric: 2*|f|*8 B per 1-D sweep / time): a fused or merged launch books
    # an equal share of its time on each sweep it performs, so these exceed the HBM peak by the fusion factor
    sweeps = {}
    names = [f"x{a + 1}" for a in range(cfg["dim_x"])] + [f"v{a + 1}" for a in range(cfg["dim_v"])]
    for a, (n, ms) in enumerate(axes):
        if n:
            gbs = sweep_bytes(cfg) / (ms / n * 1e-3) / 1e9
            sweeps[names[a]] = {"sweeps": n, "ms_share": ms / n, "effective_gbs": gbs}
    # dominant kernel = the sweep kind with the largest share of the step
    kn, (kl, kms) = max(passes.items(), key=lambda kv: kv[1][1])
    achieved = pass_bytes / (kms / kl * 1e-3) / 1e9
    tr = ncu_traffic(cfg["name"], kn)
    roofline = {"bound": "hbm", "kernel": kn, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": tr.get("traffic_bytes_per_launch") if tr else None,
                "traffic_source": (tr.get("source") if tr else None),
                "algorithmic_bytes_per_launch": pass_bytes, "peak_source": peak_src,
                "launches": kl, "avg_ms": kms / kl,
                "timed_by": "CUDA events around every launch, K steps run right after the timed region",
                "share_of_step": kms / sum(v[1] for v in kinds.values())}
    # the kernel FURTHEST below the roofline among the launch kinds that move f (>= 2 % of the step), and every kind's fraction
    total_ms = sum(v[1] for v in kinds.values())
    big = {k: v for k, v in kernels.items() if v["avg_ms"] * v["launches"] >= 0.02 * total_ms} or kernels
    wk = min(big, key=lambda k: big[k]["frac_of_measured_peak"])
    roofline["worst"] = {"kernel": wk, "frac": kernels[wk]["frac_of_measured_peak"], "avg_ms": kernels[wk]["avg_ms"],
                         "launches": kernels[wk]["launches"], "achieved": kernels[wk]["physical_gbs"],
                         "share_of_step": kernels[wk]["avg_ms"] * kernels[wk]["launches"] / total_ms}
    roofline["parts_frac"] = {k: round(v["frac_of_measured_peak"], 4) for k, v in kernels.items()}
    roofline["parts_ms_per_step"] = {k: round(v["avg_ms"] * v["launches"] / steps, 4) for k, v in kernels.items()}
    roofline["peak_is"] = ("device-to-device copy rate (read + write): kernels that mostly read, or stream with TMA, "
                           "can exceed it (frac up to ~1.08 measured)")
    parts = {k: {"launches": n, "ms_per_step": ms / steps} for k, (n, ms) in kinds.items() if n}
    res = {"workload": cfg["name"], "values": nf, "bytes_f": nf * ESIZE, "ms_per_step": ms_step,
           "single_step_ms": ms_single_calls, "step_to_ms": ms_step_to,
           "effective_gbs_per_sweep": bytes_step / (ms_step * 1e-3) / 1e9,
           "passes_per_step": n_pass / steps, "rho_passes_per_step": n_rho / steps,
           "physical_bytes_per_step": phys_step, "physical_gbs": phys_step / (ms_step * 1e-3) / 1e9,
           "physical_frac": phys_step / (ms_step * 1e-3) / 1e9 / peak,
           "kernels": kernels, "sweeps_effective": sweeps, "parts": parts, "roofline": roofline, "clocks": clocks,
           "gpu_launches": launches, "steps": steps}
    return res, ms_total_local, bytes_step * steps, g, f


def run_ours(args, cfg, rank, world, local):
    global ESIZE
    import torch
    import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SLDG path has no CPU fallback (use --impl reference "
                         "to time the CPU oracle)")
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    res, ms_total_local, bytes_local, g, f = measure_config(args, cfg, dev, local, args.steps, args.warmup, True)
    ms_total, bytes_all = aggregate(ms_total_local, bytes_local, device=dev)
    ms_step = ms_total / args.steps
    value = bytes_all / (ms_total * 1e-3) / 1e9
    peak, _ = measured_peak()
    nf, dt = res["values"], cfg["dt"]
    parts = res["parts"]
    # the paper's own figure: F * sizeof(fp) * dof / time per step, F = 20 for 3x3v and 14 otherwise,
    # where its step holds a second rho/E evaluation for the diagnostics: one measured rho pass and one
    # field solve are added to our step time.  Context only (the paper: 727 GB/s on A100 for 2x3v fp64, 626 GB/s for 3x3v).
    F = 20 if (cfg["dim_x"], cfg["dim_v"]) == (3, 3) else 14
    extra_ms = (parts.get("rho", {}).get("ms_per_step", 0.0) + parts.get("poisson", {}).get("ms_per_step", 0.0))
    paper_style = {"F": F, "gbs": F * ESIZE * nf / ((ms_step + extra_ms) * 1e-3) / 1e9 * world,
                   "ms_per_step_with_diagnostic_pass": ms_step + extra_ms,
                   "note": "PAPER.md:201-203 formula, with one more rho pass + field solve per step as in the paper's step"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": cfg["name"], "values": nf, "bytes_f": nf * ESIZE, "sweeps_per_step": sweeps_per_step(cfg),
                   "dt": dt, "poisson": args.poisson,
                   "steps_api": "sldg_steps: K Strang steps in one call, bit-identical to K sldg_step calls; the x half "
                                "steps of consecutive steps share one pass, so f at the intermediate integer "
                                "times is not written out (no per-step diagnostics inside the timed region)",
                   "l2": "inputs larger than L2 (no flush needed)" if nf * ESIZE > 2 * 126e6 else
                   "array fits in L2: numbers are L2-resident, launch-bound",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "value_is": "EFFECTIVE bandwidth per 1-D sweep (BASELINE.json metric): sweeps_per_step * 2*|f|*8 B / step time; fused "
                    "and merged passes perform several sweeps per trip over f, so it exceeds the HBM peak. The bytes the "
                    "HBM really moves are physical_bytes_per_step; physical_frac is their rate over the measured copy rate",
        "pct_of_measured_peak": 100 * value / world / peak, "pct_of_nominal_8TBs": 100 * value / world / NOMINAL_HBM_GBS,
        "physical_bytes_per_step": res["physical_bytes_per_step"], "physical_gbs": res["physical_gbs"],
        "physical_frac": res["physical_frac"], "passes_per_step": res["passes_per_step"],
        "single_step_calls": {"ms_per_step": res["single_step_ms"], "note": "K separate sldg_step calls, each ending in the caller's buffer",
                              "step_to_ms_per_step": res["step_to_ms"],
                              "step_to_note": "K sldg_step_to calls ping-ponging between f and the workspace buffer: f(t_n) after every step"},
        "paper_style": paper_style,
        "kernels": res["kernels"], "sweeps_effective": res["sweeps_effective"], "parts": parts, "roofline": res["roofline"],
        "clocks": res["clocks"], "gpu_launches": res["gpu_launches"],
    }

    # end to end through the C-ABI with HOST buffers (sldg_step_host): H2D of f, one Strang step, D2H of f, per step
    bytes_step = sweeps_per_step(cfg) * sweep_bytes(cfg)
    if rank == 0 or world > 1:
        try:
            fh = torch.empty(g.shape, dtype=f.dtype, pin_memory=True)
            fh.copy_(f)
            nrep = max(1, min(args.steps, 2 if nf * ESIZE > 2e10 else 3))
            g.step_host(fh, f, dt, nsteps=1)                    # warm-up
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            for _ in range(nrep):
                g.step_host(fh, f, dt, nsteps=1)
            torch.cuda.synchronize(dev)
            e2e_ms_local = 1e3 * (time.perf_counter() - t0)
            e2e_ms, e2e_bytes = aggregate(e2e_ms_local, bytes_step * nrep, device=dev)
            line["e2e"] = {"value": e2e_bytes / (e2e_ms * 1e-3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": nf * ESIZE,
                           "d2h_bytes_per_step": nf * ESIZE, "ms_per_step": e2e_ms / nrep, "steps": nrep,
                           "api": "sldg_step_host (pinned host f -> device, 1 Strang step, device -> host)"}
            del fh
        except Exception as ex:                                  # e.g. not enough pinned host memory
            line["e2e"] = {"value": None, "unit": UNIT, "error": str(ex)[:200]}

    # the other BASELINE.json configs, briefly, in the same invocation (rank 0, single GPU): one block per config
    if rank == 0 and world == 1 and args.all_configs and not args.workload and not args.cells:
        g.close()
        del g, f
        torch.cuda.empty_cache()
        others = {}
        for i, oc in enumerate(W.CONFIGS):
            if oc["name"] == cfg["name"]:
                continue
            try:
                r, _, _, g2, f2 = measure_config(args, oc, dev, local, min(args.steps, 10), 3, False)
                g2.close()
                del g2, f2
                torch.cuda.empty_cache()
                rf = r["roofline"]
                others[oc["name"]] = {"ms_per_step": r["ms_per_step"], "single_step_ms": r["single_step_ms"], "step_to_ms": r["step_to_ms"],
                                      "effective_gbs_per_sweep": r["effective_gbs_per_sweep"],
                                      "passes_per_step": r["passes_per_step"],
                                      "physical_bytes_per_step": r["physical_bytes_per_step"],
                                      "physical_gbs": r["physical_gbs"], "physical_frac": r["physical_frac"],
                                      "roofline": {"kernel": rf["kernel"], "frac": rf["frac"], "avg_ms": rf["avg_ms"],
                                                   "achieved": rf["achieved"], "worst": rf["worst"]},
                                      "kernels": {k: {"avg_ms": v["avg_ms"], "frac_of_measured_peak": v["frac_of_measured_peak"],
                                                      "launches": v["launches"]} for k, v in r["kernels"].items()},
                                      "clocks": r["clocks"], "steps": r["steps"],
                                      "note": "L2-resident, launch-bound" if r["bytes_f"] < 2 * 126e6 else ""}
            except Exception as ex:
                others[oc["name"]] = {"error": str(ex)[:200]}
        line["configs"] = others
        # NEXT rows, driver-measured: the paper's default order (k = 3) on the two bump-on-tail workloads, and the
        # headline config in single precision (Tables 3-4)
        import argparse as _ap
        nxt = {c["name"]: c for c in W.NEXT_CONFIGS}
        legs = [("bot_6d_k3_9", nxt.get("bot_6d_k3_9"), "f64"), ("bot_5d_k3_16", nxt.get("bot_5d_k3_16"), "f64"),
                (cfg["name"] + "_f32", cfg, "f32")]
        f32 = {}
        for name, oc, prec in legs:
            if oc is None or args.dtype != "f64":
                continue
            a2 = _ap.Namespace(**vars(args))
            a2.dtype = prec
            es0, ESIZE = ESIZE, (4 if prec == "f32" else 8)
            try:
                r, _, _, g2, f2 = measure_config(a2, oc, dev, local, min(args.steps, 10), 3, False)
                g2.close()
                del g2, f2
                torch.cuda.empty_cache()
                blk = {"ms_per_step": r["ms_per_step"], "single_step_ms": r["single_step_ms"], "step_to_ms": r["step_to_ms"], "dtype": prec,
                       "passes_per_step": r["passes_per_step"], "physical_gbs": r["physical_gbs"],
                       "physical_frac": r["physical_frac"], "effective_gbs_per_sweep": r["effective_gbs_per_sweep"],
                       "worst": r["roofline"]["worst"], "parts_frac": r["roofline"]["parts_frac"],
                       "parts_ms_per_step": r["roofline"]["parts_ms_per_step"], "steps": r["steps"]}
            except Exception as ex:
                blk = {"error": str(ex)[:200]}
            finally:
                ESIZE = es0
            if prec == "f32":
                f32[name] = blk
            else:
                others[name] = blk
        if f32:
            line["f32"] = f32
        # one compact row per config INSIDE the roofline block (the driver's record keeps that block whole):
        # [ms_per_step, passes_per_step, physical_frac, worst kernel, its frac]
        def row(r):
            w = r.get("worst") or (r.get("roofline") or {}).get("worst") or {}
            return [round(r["ms_per_step"], 4), r["passes_per_step"], round(r["physical_frac"], 4), w.get("kernel"),
                    round(w.get("frac", 0.0), 4), round(r["single_step_ms"], 4), round(r["step_to_ms"], 4)] if "ms_per_step" in r else [r.get("error")]
        line["roofline"]["by_config"] = {n: row(r) for n, r in list(others.items()) + list(f32.items())}
        line["roofline"]["by_config_columns"] = "ms_per_step (sldg_steps), passes_per_step, physical_frac, worst kernel, worst frac, ms per sldg_step call, ms per sldg_step_to call"
        line["roofline"]["headline_single_step_ms"] = [round(res["single_step_ms"], 4), round(res["step_to_ms"], 4)]
        line["roofline"]["previous_round_headline"] = "cfg5_6d_twostream_24x20_k1 (round 2: 72.29 ms; round 1 headline was cfg2)"

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        r = time_oracle(cfg, steps=1000, warmup=1, budget_s=12.0)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "ms_per_step")}
        r1 = time_oracle(cfg, steps=1000, warmup=0, budget_s=8.0, threads=1)
        line["cpu_baseline"]["single_thread"] = {k: r1[k] for k in ("value", "unit", "cores", "ms_per_step", "sample")}
    return line if rank == 0 else None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs (default 4: cfg5, the largest "
                    "single-GPU configuration, 56.6 GB + as much workspace)")
    ap.add_argument("--no-all-configs", dest="all_configs", action="store_false", help="skip the brief runs of the other "
                    "BASELINE.json configs that the default run attaches under `configs`")
    ap.add_argument("--workload", type=str, default=None, help="a workload by name, incl. the NEXT-row cases "
                    "(bot_5d_k3_16, bot_6d_k3_9: the paper's bump-on-tail case, 4th order)")
    ap.add_argument("--cfl", type=float, default=None, help="choose dt so that the largest x shift is CFL cells (PAPER.md:351)")
    ap.add_argument("--poisson", default="fft", choices=["fft", "cg"], help="field solver inside the step: the FFT "
                    "route (default) or the CGdG solver with the paper's tolerance 1e-3 and warm start (PAPER.md:496-567)")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"], help="f32: single precision mode (PAPER.md:191); "
                    "the metric then counts 2*|f|*4 B per sweep")
    ap.add_argument("--option", action="append", default=None, help="a tuning knob of sldg_set_option as name=value (repeatable), "
                    "e.g. --option x_double=2 (profiles/ uses this to capture kernels the default plan does not launch)")
    ap.add_argument("--cells", type=str, default=None, help="override cells, e.g. 16,16,16,16 (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    import workloads as W
    global ESIZE
    ESIZE = 4 if args.dtype == "f32" else 8
    cfg = W.CONFIGS[args.config]
    if args.workload:
        cfg = {c["name"]: c for c in W.CONFIGS + W.NEXT_CONFIGS}[args.workload]
    if args.cfl:
        cfg = W.with_cfl(cfg, args.cfl)
    if args.cells:
        cfg = W.scaled(cfg, [int(c) for c in args.cells.split(",")])
    if args.impl == "reference":
        rank = int(os.environ.get("RANK", "0"))
        line = run_reference(args, cfg, rank, int(os.environ.get("WORLD_SIZE", "1")))
    else:
        rank, world, local = dist_setup(args.gpus)
        line = run_ours(args, cfg, rank, world, local)
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
