#!/usr/bin/env python
"""bench.py — HOMG solve throughput on B200 (driver contract: one JSON line on stdout from rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

A "step" is one whole solve of the workload: reset u <- u0, c* outer HOMG cycles (residual ->
restriction -> MFMG visits -> u += e; c* = cycles the solve needs to reach the config's relative
residual, found once during warm-up from the device-side norm history), and the final residual norm.
  value        fine-grid unknowns solved per second, inputs resident in HBM (device-timed, CUDA events)
  e2e          the same through the C ABI with HOST buffers (pinned): H2D of f and u0, the solve, D2H of u
  roofline     the dominant kernel (level-0 Jacobi sweep), timed live with CUDA events per launch
  cpu_baseline the oracle (oracle/, Algorithm H, single thread) on a bounded sample of the same solve
N > 1: independent replicas, one per GPU ("replicas only": the path has no exchange step).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1108_2045_b200 import inputs as I  # noqa: E402

METRIC = "fine-grid unknowns/s (time to the config's relative residual)"
UNIT = "unknowns/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="homg", choices=["homg", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(I.CONFIGS))
    ap.add_argument("--n", type=int, default=0, help="scale the workload to an n^d grid (debugging)")
    ap.add_argument("--cycle", default="mfmg", choices=["mfmg", "v", "literal"],
                    help="mfmg: the paper's HOMG cycle (default); v: classic V(2,1) on the same kernels; "
                         "literal: the paper's own whole-grid design (one fine array, one launch per iteration)")
    ap.add_argument("--mixed", action="store_true",
                    help="mixed-precision outer loop (SURVEY.md 8(f)2): u, f, residual in fp64, the correction cycle in "
                         "fp32; the workload's inputs are generated in fp64 (cfg3/cfg4: makes tolerances below the "
                         "fp32 floor reachable; cfg2/cfg5: halves the sweep traffic)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the largest-3-D-grid roofline pass")
    ap.add_argument("--cpu-seconds", type=float, default=20.0)
    return ap.parse_args()


def workload_config(cfg):
    return {"workload": f"{cfg.name}: {'x'.join(map(str, cfg.dims))} nodes, {cfg.dtype}, {cfg.levels} levels, "
                        f"{cfg.stencil}, omega={cfg.omega:.6g}, MFMG schedule C MaxI={cfg.max_iters}, "
                        f"stop rel. residual {cfg.tol:g}" if cfg.tol > 0 else
                        f"{cfg.name}: {'x'.join(map(str, cfg.dims))} nodes, {cfg.dtype}, {cfg.levels} levels, "
                        f"{cfg.stencil}, omega={cfg.omega:.6g}, MFMG schedule C MaxI={cfg.max_iters}, {cfg.cycles} cycles",
            "dims": list(cfg.dims), "levels": cfg.levels, "stencil": cfg.stencil, "tol": cfg.tol,
            "parallelism": "replicas only (one independent solve per GPU)"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons, sampled while the timed regions run."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.marks, self.proc = [], [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def mark(self, t0, t1):
        self.marks.append((t0, t1))

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if any(a - 0.05 <= t <= b + 0.05 for a, b in self.marks)] or \
               [r for (_, r) in self.rows]
        sm, reasons, mx = [], set(), None
        for r in rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def cycles_to_tol(hist_plus_final, cfg):
    """first c such that ||r_c|| / ||r_0|| <= tol (norm BEFORE cycle c == after cycle c-1); fixed count if tol == 0."""
    if cfg.tol <= 0:
        return cfg.cycles, None
    n0 = hist_plus_final[0]
    for c, v in enumerate(hist_plus_final):
        if v <= cfg.tol * n0:
            return c, v / n0
    return None, min(hist_plus_final) / n0


def make_solver(cfg, inp, torch, dev, vcycle=None, literal=False, mixed=False):
    from paper_1108_2045_b200 import homg
    s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, cfg.dtype, omega=cfg.omega, max_iters=cfg.max_iters,
                    schedule=cfg.schedule, device=dev, vcycle=vcycle, literal=literal, mixed=mixed)
    tdt = torch.float64 if cfg.dtype == "f64" else torch.float32
    d = {k: (None if v is None else torch.from_numpy(v).to(dev)) for k, v in inp.items()}
    if not inp["u0"].any():
        d["u0"] = None          # the config's u0 = 0 is the library's default guess: set_initial_guess(None), no array
    if d["k"] is not None:
        s.set_coefficient(d["k"])
    s.set_rhs(d["f"])
    s.set_initial_guess(d["u0"])
    return s, d, tdt


def find_cstar(s, d, cfg):
    """runs the capped cycle count once and reads the history back (outside any timed region)."""
    s.set_initial_guess(d["u0"])
    s.cycle(cfg.cycles)
    hist = s.residual_history()
    final, _ = s.residual_norm()
    c, rel = cycles_to_tol(hist + [final], cfg)
    stagnated = c is None
    if stagnated:      # tolerance below the arithmetic's floor (R17): stop where the norm stops falling
        allv = hist + [final]
        c = int(np.argmin(allv))
    return max(1, c), rel, stagnated, (hist + [final])


# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from `ncu --set full`
# captures, one launch each; the summaries and their commands are under profiles/.
NCU_TRAFFIC = {
    ("cfg4", "visit_l0"): (1.318703e9 + 0.514103e9, "profiles/r01e_ncu_full_cfg4.md"),
    ("cfg4", "residual_l0"): (1.152890e9 + 0.571569e9, "profiles/r01e_ncu_full_cfg4.md"),
    ("cfg4", "relax_l0"): (1.164186e9 + 0.509018e9, "profiles/r01b_ncu_full_cfg4.md"),
    ("cfg2", "visit_l0"): (43.483904e6 + 0.012800e6, "profiles/r01d_ncu_full_cfg2.md"),      # L2-resident (17 MB arrays)
    ("cfg2", "residual_l0"): (36.909056e6 + 0.042752e6, "profiles/r01d_ncu_full_cfg2.md"),
    ("cfg3", "visit_l0"): (693.390848e6 + 235.526656e6, "profiles/r01e_ncu_full_cfg3.md"),
    ("cfg3", "residual_l0"): (548.102656e6 + 302.414592e6, "profiles/r01e_ncu_full_cfg3.md"),
    ("cfg5", "relax_l0"): (687.057920e6 + 121.797120e6, "profiles/r01e_ncu_full_cfg5.md"),
    ("cfg5", "relax_l0_last"): (821.715712e6 + 122.345984e6, "profiles/r01e_ncu_full_cfg5.md"),
    ("cfg5", "residual_l0"): (690.258176e6 + 137.026304e6, "profiles/r01e_ncu_full_cfg5.md"),
}
LEVEL0_CLASSES = ("visit_l0", "relax_l0", "relax_l0_first", "relax_l0_last", "residual_l0")


def roofline_from_profile(prof, peak, peak_src, comp=None, cycles=1, wname=""):
    """roofline of the level-0 kernel class that takes the most time (K_visit = the fused
    interpolate+correct+relax visit when it runs): achieved = ALGORITHMIC bytes (3 arrays
    per Jacobi node-update, (2+2/2^d) for the first sweep of a visit, 4 for the one that adds u) over the
    event-timed duration.  K_visit performs the sweeps of a visit in one pass, so its COMPULSORY bytes
    (what the launch itself must move) are reported next to it; `traffic` is the ncu DRAM byte count."""
    if not prof:
        return None, {}
    comp = comp or {}
    total_ms = sum(v[0] for v in prof.values())
    l0 = [k for k in prof if k in LEVEL0_CLASSES]
    name = max(l0 or prof, key=lambda k: prof[k][0])
    shares = {}
    for k, v in prof.items():
        cb = comp.get(k, 0.0) * cycles
        shares[k] = {"ms_per_launch": v[0] / v[1], "launches": v[1], "share": v[0] / total_ms,
                     "algorithmic_gbs": (v[2] / (v[0] * 1e-3) / 1e9) if v[0] > 0 else 0.0,
                     "compulsory_gbs": (cb / (v[0] * 1e-3) / 1e9) if v[0] > 0 else 0.0}
    ms, cnt, by = prof[name]
    ach = by / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
    cb = comp.get(name, 0.0) * cycles
    tr = NCU_TRAFFIC.get((wname, name))
    rl = {"bound": "hbm", "kernel": name, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
          "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None,
          "peak_source": peak_src, "ms_per_launch": ms / cnt, "launches": cnt,
          "bytes_per_launch": by / cnt, "compulsory_bytes_per_launch": cb / cnt,
          "compulsory_gbs": cb / (ms * 1e-3) / 1e9 if ms > 0 else 0.0,
          "share_of_cycle": ms / total_ms, "frac_of_8TBs_nominal": ach / 8000.0,
          "note": "achieved counts the per-sweep algorithmic bytes of SURVEY.md 8(d); a fused multi-sweep "
                  "launch (visit_l0) moves only compulsory_bytes_per_launch, so achieved may exceed the HBM peak"}
    return rl, shares


def cpu_baseline(cfg, inp, cstar, seconds):
    """the oracle as it stands (Algorithm H, one thread) on the first cycles of the same solve."""
    from oracle import oracle as O
    sched = O.schedule(cfg.schedule, cfg.levels, cfg.max_iters)
    u = inp["u0"].copy()
    t_used, ncyc = 0.0, 0
    while ncyc < cstar and (ncyc == 0 or t_used + t_used / ncyc <= seconds):
        t0 = time.perf_counter()
        u, _, _ = O.homg("H", inp["f"], u, cfg.levels, cfg.omega, sched, 1, k=inp["k"], keep_history=False)
        t_used += time.perf_counter() - t0
        ncyc += 1
    t_cycle = t_used / ncyc
    return {"value": cfg.n_interior / (t_cycle * cstar), "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"first {ncyc} of {cstar} cycles of the same solve ({t_used:.1f} s), scaled to {cstar} cycles",
            "s_per_cycle": t_cycle, "host_cores_available": os.cpu_count()}


def run_reference(args):
    """--impl reference: the oracle (CPU, one thread) on the same workload.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import oracle as O
    cfg = I.CONFIGS[args.workload]
    if args.n:
        cfg = I.scaled(cfg, args.n)
    inp = I.make_inputs(cfg)
    sched = O.schedule(cfg.schedule, cfg.levels, cfg.max_iters)
    budget = 150.0
    # warm-up: cycles until the tolerance (bounded) -> c*; t_cycle estimate
    t0 = time.perf_counter()
    u = inp["u0"].copy()
    norms, cstar = [], None
    for c in range(cfg.cycles):
        u, _, n = O.homg("H", inp["f"], u, cfg.levels, cfg.omega, sched, 1, k=inp["k"], keep_history=False)
        if c == 0:
            norms.append(n[0])
        norms.append(n[1])
        if cfg.tol > 0 and n[1] <= cfg.tol * norms[0]:
            cstar = c + 1
            break
        if time.perf_counter() - t0 > budget / 3:
            break
    done = len(norms) - 1
    t_cycle0 = (time.perf_counter() - t0) / done
    known = {"cfg2": 14, "cfg3": 7, "cfg4": 9, "cfg5": 20}      # SURVEY.md A.2 probe counts, used only if the
    if cstar is None:                                           # bounded warm-up did not reach the tolerance
        cstar = cfg.cycles if cfg.tol <= 0 else known.get(cfg.name.split("@")[0], done)
    per_step = max(1, min(cstar, int((budget * 2 / 3) / max(1, args.steps) / t_cycle0)))
    t_sum = 0.0
    for _ in range(args.steps):
        u = inp["u0"].copy()
        t1 = time.perf_counter()
        O.homg("H", inp["f"], u, cfg.levels, cfg.omega, sched, per_step, k=inp["k"], keep_history=False)
        t_sum += time.perf_counter() - t1
    t_cycle = t_sum / (args.steps * per_step)
    t_solve = t_cycle * cstar
    val = cfg.n_interior / t_solve
    sample = f"{per_step} of {cstar} cycles per step, scaled to {cstar} cycles"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_solve * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic", "config": workload_config(cfg),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "cycles_to_tol": cstar, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_homg(args):
    import torch
    import torch.distributed as dist
    from paper_1108_2045_b200 import replicas
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    rank, world = replicas.init("nccl", torch.device(dev))
    cfg = I.CONFIGS[args.workload]
    if args.n:
        cfg = I.scaled(cfg, args.n)
    if args.mixed:
        import dataclasses
        cfg = dataclasses.replace(cfg, dtype="f64")
    inp = I.make_inputs(cfg)
    s, d, _ = make_solver(cfg, inp, torch, dev, vcycle=(2, 1) if args.cycle == "v" else None,
                          literal=args.cycle == "literal", mixed=args.mixed)
    cstar, rel, stagnated, norms = find_cstar(s, d, cfg)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    sampler = ClockSampler(local)
    stream = torch.cuda.current_stream()

    def step_dev():
        s.set_initial_guess(d["u0"])
        s.cycle(cstar)
        return s.residual_norm()

    def sync_all():
        torch.cuda.synchronize()
        replicas.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        flush.zero_()
        step_dev()
    sync_all()
    t_a = time.time()
    total_ms = 0.0
    for _ in range(args.steps):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        final = step_dev()
        e1.record(stream)
        e1.synchronize()
        total_ms += e0.elapsed_time(e1)
    sync_all()
    sampler.mark(t_a, time.time())

    # ---- e2e: host buffers through the C ABI ----
    hf = torch.from_numpy(inp["f"]).pin_memory()
    hu0 = torch.from_numpy(inp["u0"]).pin_memory() if inp["u0"].any() else None     # u0 = 0: the default guess, no upload
    hk = None if inp["k"] is None else torch.from_numpy(inp["k"]).pin_memory()
    hout = torch.empty(cfg.dims, dtype=hf.dtype).pin_memory()

    def step_e2e():
        if hk is not None:
            s.set_coefficient(hk)
        s.set_rhs(hf)
        s.set_initial_guess(hu0)
        s.cycle(cstar)
        r = s.residual_norm()
        s.get_solution(hout)
        return r

    for _ in range(2):
        step_e2e()
    sync_all()
    t_b = time.time()
    e2e_s = 0.0
    n_e2e = max(1, min(args.steps, 10))
    for _ in range(n_e2e):
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        step_e2e()
        torch.cuda.synchronize()
        e2e_s += time.perf_counter() - t0
    sync_all()
    sampler.mark(t_b, time.time())

    # ---- per-kernel timing (CUDA events after every launch, plain stream launches) ----
    prof = {}
    if not args.mixed:                          # (homg_profile_cycles is not available in mixed precision)
        s.set_initial_guess(d["u0"])
        s.profile_cycles(1)                     # warm
        s.set_initial_guess(d["u0"])
        t_c = time.time()
        prof = s.profile_cycles(cstar)
        sampler.mark(t_c, time.time())
    peak, peak_src = peaks()
    comp, comp_total = s.compulsory_bytes_per_cycle()
    rl, shares = roofline_from_profile(prof, peak, peak_src, comp, cstar, cfg.name)
    launches_step = s.launches_per_cycle() * cstar + (2 if d["u0"] is not None else 0) + 2   # + pack(u0) (u0 = 0: a memset, not counted) + norm-only pass (2 kernels)
    bytes_cycle = s.bytes_per_cycle()
    clocks = sampler.stop()

    total_ms, e2e_s = replicas.max_over_ranks([total_ms, e2e_s], device=dev)
    es = 8 if cfg.dtype == "f64" else 4
    nbytes = int(np.prod(cfg.dims)) * es
    line = {"metric": METRIC, "value": replicas.job_value(cfg.n_interior, args.steps, world, total_ms), "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 (u, f, residual) / f32 (correction cycle)" if args.mixed else cfg.dtype, "data": "synthetic",
            "config": dict(workload_config(cfg), l2="flushed between steps (512 MiB write)",
                           cycle={"mfmg": "MFMG (HOMG), per-level arrays", "v": "classic V(2,1)",
                                  "literal": "MFMG (HOMG), paper-literal whole-grid iteration"}[args.cycle]),
            "cycles_to_tol": cstar, "rel_residual_reached": float(final[1]), "stagnated_above_tol": bool(stagnated),
            "ms_per_cycle": total_ms / args.steps / cstar,
            "unknowns_per_s_per_cycle": cfg.n_interior * world / (total_ms * 1e-3 / args.steps / cstar),
            "cycle_algorithmic_gb": bytes_cycle / 1e9,
            "cycle_algorithmic_gbs": bytes_cycle / (total_ms * 1e-3 / args.steps / cstar) / 1e9,
            "cycle_compulsory_gb": comp_total / 1e9,
            "cycle_compulsory_gbs": comp_total / (total_ms * 1e-3 / args.steps / cstar) / 1e9,
            "e2e": {"value": cfg.n_interior * n_e2e * world / e2e_s, "unit": UNIT, "ms_per_step": e2e_s / n_e2e * 1e3,
                    "h2d_bytes_per_step": nbytes * (1 + (hk is not None) + (hu0 is not None)), "d2h_bytes_per_step": nbytes + 8},
            "gpu_launches": launches_step * args.steps, "roofline": rl, "kernels": shares, "clocks": clocks}
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(cfg, inp, cstar, args.cpu_seconds)
        if not args.no_extra and world == 1 and not args.n and args.workload != "cfg4" and not args.mixed:
            line["roofline_largest_3d"] = extra_largest(torch, dev, peak, peak_src)
        if not args.no_extra and world == 1 and args.cycle == "mfmg" and not args.mixed:
            line["classic_v21"] = extra_other(torch, dev, cfg, inp, flush, vcycle=(2, 1))
            line["paper_literal"] = extra_other(torch, dev, cfg, inp, flush, literal=True)
        print(json.dumps(line), flush=True)
    s.destroy()
    if world > 1:
        dist.destroy_process_group()


def extra_other(torch, dev, cfg, inp, flush, vcycle=None, literal=False):
    """the same solve with another cycle on the same hierarchy and operators: the classic V(2,1) cycle — the
    comparison the paper argues — or the paper's own whole-grid design (Algorithm L:
    one fine-grid array, one whole-grid launch per iteration, L51/L119), which the per-level layout replaces."""
    s, d, _ = make_solver(cfg, inp, torch, dev, vcycle=vcycle, literal=literal)
    cstar, rel, stagnated, _ = find_cstar(s, d, cfg)
    reps = 2 if literal else 5
    for _ in range(1 if literal else 3):
        s.set_initial_guess(d["u0"]); s.cycle(cstar); s.residual_norm()
    ms = 0.0
    for _ in range(reps):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        s.set_initial_guess(d["u0"]); s.cycle(cstar); fin = s.residual_norm()
        e1.record(); e1.synchronize()
        ms += e0.elapsed_time(e1)
    ms /= reps
    out = {"cycles_to_tol": cstar, "ms_per_step": ms, "ms_per_cycle": ms / cstar, "value": cfg.n_interior / (ms * 1e-3),
           "unit": UNIT, "rel_residual_reached": float(fin[1]), "stagnated_above_tol": bool(stagnated),
           "launches_per_cycle": s.launches_per_cycle()}
    s.destroy()
    return out


def extra_largest(torch, dev, peak, peak_src):
    """north_star's bandwidth target is quoted on the largest 3-D grid (cfg4, 513^3 fp32): per-kernel
    event timing of a few cycles there (arrays of 540 MB, far larger than L2)."""
    cfg = I.CONFIGS["cfg4"]
    inp = I.make_inputs(cfg)
    s, d, _ = make_solver(cfg, inp, torch, dev)
    s.cycle(2)
    torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record(); s.cycle(5); e1.record(); e1.synchronize()
    ms_cycle = e0.elapsed_time(e1) / 5
    prof = s.profile_cycles(3)
    comp, _ = s.compulsory_bytes_per_cycle()
    rl, shares = roofline_from_profile(prof, peak, peak_src, comp, 3, cfg.name)
    out = {"workload": workload_config(cfg)["workload"], "ms_per_cycle_graph": ms_cycle,
           "unknowns_per_s_per_cycle": cfg.n_interior / (ms_cycle * 1e-3),
           "cycle_algorithmic_gbs": s.bytes_per_cycle() / (ms_cycle * 1e-3) / 1e9, "dominant": rl, "kernels": shares}
    s.destroy()
    return out


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_homg(a)
