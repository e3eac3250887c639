#!/usr/bin/env python
"""bench.py — HOMG solve throughput on B200 (driver contract: one JSON line on stdout from rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl reference]

A "step" is one whole solve of the workload through homg_solve: reset u <- u0, then outer HOMG cycles
(residual -> restriction -> MFMG visits -> u += e) repeated ON THE DEVICE until the config's relative residual
is reached — the cycle count is decided by the solve itself, not learnt beforehand.
  value        fine-grid unknowns solved per second, inputs resident in HBM (device-timed, CUDA events)
  e2e          the same through the C ABI with HOST buffers (pinned): H2D of f (u0, k), the solve, D2H of u
  roofline     the level-0 kernel class with the largest share of the cycle, timed live with CUDA events per launch;
               achieved = the bytes the launch itself must move / its duration
  cpu_baseline the oracle (oracle/, Algorithm H, single thread, untuned) on a bounded sample of the same workload
Default workload: cfg4 (513^3 fp32, 540 MB per array — HBM-resident; north_star quotes its bandwidth target on
it).  N > 1: independent replicas, one per GPU ("replicas only": the path has no exchange step).
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
    ap.add_argument("--workload", default="cfg4", choices=sorted(I.CONFIGS))
    ap.add_argument("--n", type=int, default=0, help="scale the workload to an n^d grid (debugging)")
    ap.add_argument("--cycle", default="mfmg", choices=["mfmg", "v", "literal"],
                    help="mfmg: the paper's HOMG cycle (default); v: classic V(2,1) on the same kernels; "
                         "literal: the paper's own whole-grid design (one fine array, one launch per iteration)")
    ap.add_argument("--mixed", action="store_true",
                    help="mixed-precision outer loop (SURVEY.md 8(f)2): u, f, residual in fp64, the correction cycle in "
                         "fp32; the workload's inputs are generated in fp64 (cfg3/cfg4: makes tolerances below the "
                         "fp32 floor reachable; cfg2/cfg5: halves the sweep traffic)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the side rows (classic V(2,1), paper-literal mode)")
    ap.add_argument("--cpu-seconds", type=float, default=20.0)
    ap.add_argument("--ref-seconds", type=float, default=120.0, help="--impl reference: budget of the whole run")
    return ap.parse_args()


def workload_config(cfg, cycle="mfmg"):
    stop = f"stop rel. residual {cfg.tol:g}" if cfg.tol > 0 else f"{cfg.cycles} cycles"
    return {"workload": f"{cfg.name}: {'x'.join(map(str, cfg.dims))} nodes, {cfg.dtype}, {cfg.levels} levels, "
                        f"{cfg.stencil}, omega={cfg.omega:.6g}, MFMG schedule C MaxI={cfg.max_iters}, {stop}",
            "dims": list(cfg.dims), "levels": cfg.levels, "stencil": cfg.stencil, "tol": cfg.tol,
            "parallelism": "replicas only (one independent solve per GPU)",
            "l2": "flushed between steps (512 MiB write); level-0 arrays of cfg3-5 are larger than L2",
            "cycle": {"mfmg": "MFMG (HOMG), per-level arrays", "v": "classic V(2,1)",
                      "literal": "MFMG (HOMG), paper-literal whole-grid iteration"}[cycle]}


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


def make_solver(cfg, inp, torch, dev, vcycle=None, literal=False, mixed=False):
    from paper_1108_2045_b200 import homg
    s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, cfg.dtype, omega=cfg.omega, max_iters=cfg.max_iters,
                    schedule=cfg.schedule, device=dev, vcycle=vcycle, literal=literal, mixed=mixed)
    d = {k: (None if v is None else torch.from_numpy(v).to(dev)) for k, v in inp.items()}
    if not inp["u0"].any():
        d["u0"] = None          # the config's u0 = 0 is the library's default guess: set_initial_guess(None), no array
    if d["k"] is not None:
        s.set_coefficient(d["k"])
    s.set_rhs(d["f"])
    s.set_initial_guess(d["u0"])
    return s, d


class Solve:
    """one solve of the workload = one bench step.  MFMG: homg_solve (the device-side loop stops by itself; a config
    without a tolerance runs its fixed cycle count; --mixed: the mixed-precision loop, also through homg_solve).  Side
    rows (classic V, paper-literal) have no homg_solve: they run the cycle count a first run of the same solve needed (find_cstar)."""

    def __init__(self, s, cfg, own_loop):
        self.s, self.cfg, self.own_loop, self.cstar = s, cfg, own_loop, None

    def find_cstar(self, u0):
        cfg, s = self.cfg, self.s
        s.set_initial_guess(u0)
        s.cycle(cfg.cycles)
        allv = s.residual_history() + [s.residual_norm()[0]]
        c = next((i for i, v in enumerate(allv) if v <= cfg.tol * allv[0]), None) if cfg.tol > 0 else cfg.cycles
        self.cstar = max(1, int(np.argmin(allv)) if c is None else c)
        return self.cstar

    def run(self, u0):
        """-> (cycles, final relative residual)"""
        cfg, s = self.cfg, self.s
        s.set_initial_guess(u0)
        if self.own_loop and cfg.tol > 0:
            return s.solve(cfg.tol, cfg.cycles)
        n = self.cstar if self.cstar is not None else cfg.cycles
        s.cycle(n)
        return n, s.residual_norm()[1]


# DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from `ncu --set full` captures, one launch
# each; the summaries and their commands are under profiles/ (the tag names the capture, so a stale entry shows).
NCU_TRAFFIC = {
    ("cfg4", "visit_l0"): (1.301990e9 + 0.512010e9, "profiles/r02a_ncu_full_cfg4.md"),
    ("cfg4", "residual_l0"): (1.152890e9 + 0.571569e9, "profiles/r01e_ncu_full_cfg4.md (kernel unchanged since)"),
    ("cfg3", "visit_l0"): (693.407488e6 + 234.450432e6, "profiles/r02c_ncu_full_cfg3.md"),
    ("cfg3", "residual_l0"): (548.152832e6 + 302.227200e6, "profiles/r02c_ncu_full_cfg3.md"),
    ("cfg5", "visit_l0"): ((1.005716e9 + 0.127886e9 + 0.759066e9 + 0.125065e9) / 2, "profiles/r02b_ncu_full_cfg5.md (mean of the two passes of a visit)"),
    ("cfg5", "relax_l0"): (687.057920e6 + 121.797120e6, "profiles/r01e_ncu_full_cfg5.md (kernel unchanged since; HOMG_VISIT_VAR=0)"),
    ("cfg5", "relax_l0_last"): (821.715712e6 + 122.345984e6, "profiles/r01e_ncu_full_cfg5.md (kernel unchanged since; HOMG_VISIT_VAR=0)"),
    ("cfg5", "residual_l0"): (0.690248e9 + 0.136572e9, "profiles/r02b_ncu_full_cfg5.md"),
}
LEVEL0_CLASSES = ("visit_l0", "relax_l0", "relax_l0_first", "relax_l0_last", "residual_l0")


def roofline_from_profile(prof, peak, peak_src, comp, cycles, wname):
    """Per kernel class (CUDA events after every launch, homg_profile_cycles): duration, share of the cycle and
      hbm_gbs        = the bytes the launches themselves must move ("compulsory": every array a launch reads or
                       writes, once) / duration — the HBM roofline number, frac = hbm_gbs / peak;
      sweep_equiv_gbs = SURVEY.md 8(d)'s per-sweep count (3 arrays per Jacobi node-update) / duration: equal to
                       hbm_gbs for single-operation kernels, larger for K_visit, which runs the eta sweeps of a
                       visit in one pass (it may exceed the HBM peak; it is not a bandwidth).
    `roofline` = the level-0 class with the largest share."""
    if not prof:
        return None, {}
    total_ms = sum(v[0] for v in prof.values())
    shares = {}
    for k, v in prof.items():
        cb = comp.get(k, 0.0) * cycles
        tr = NCU_TRAFFIC.get((wname, k))
        sec = v[0] * 1e-3
        shares[k] = {"ms_per_launch": v[0] / v[1], "launches": v[1], "share": v[0] / total_ms,
                     "hbm_gbs": cb / sec / 1e9 if sec > 0 else 0.0, "frac_of_peak": cb / sec / 1e9 / peak if sec > 0 else 0.0,
                     "bytes_per_launch": cb / v[1], "sweep_equiv_gbs": v[2] / sec / 1e9 if sec > 0 else 0.0,
                     "ncu_dram_bytes_per_launch": tr[0] if tr else None}
    l0 = [k for k in prof if k in LEVEL0_CLASSES]
    name = max(l0 or prof, key=lambda k: prof[k][0])
    k = shares[name]
    tr = NCU_TRAFFIC.get((wname, name))
    rl = {"bound": "hbm", "kernel": name, "achieved": k["hbm_gbs"], "peak": peak, "unit": "GB/s", "frac": k["frac_of_peak"],
          "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None, "peak_source": peak_src,
          "ms_per_launch": k["ms_per_launch"], "launches": k["launches"], "bytes_per_launch": k["bytes_per_launch"],
          "share_of_cycle": k["share"], "frac_of_8TBs_nominal": k["hbm_gbs"] / 8000.0,
          "sweep_equiv_gbs": k["sweep_equiv_gbs"],
          "note": "achieved = bytes the launch itself must move / CUDA-event duration. visit_l0 (interpolate+correct + "
                  "4 sweeps + u += e in one pass) is bound by instruction issue and shared-memory bandwidth, not by "
                  "HBM (profiles/): its frac is what is left to the HBM floor; sweep_equiv_gbs counts the per-sweep "
                  "bytes of SURVEY.md 8(d) and is not a bandwidth"}
    return rl, shares


def sample_config(cfg, seconds_per_solve):
    """the workload's recipe at the largest n^d grid (n = 2^j + 1, at most the workload's own) whose oracle solve is
    estimated to fit `seconds_per_solve`: the oracle's cost is linear in the nodes (pin P10)."""
    from oracle import oracle as O
    nd = len(cfg.dims)
    small = I.scaled(cfg, 33 if nd == 3 else 257)
    inp = I.make_inputs(small)
    sched = O.schedule(small.schedule, small.levels, small.max_iters)
    O.homg("H", inp["f"], inp["u0"], small.levels, small.omega, sched, 1, k=inp["k"], keep_history=False)     # warm
    t0 = time.perf_counter()
    O.homg("H", inp["f"], inp["u0"], small.levels, small.omega, sched, 2, k=inp["k"], keep_history=False)
    per_node_cycle = (time.perf_counter() - t0) / 2 / float(np.prod(small.dims))
    est_cycles = 12 if cfg.tol > 0 else cfg.cycles
    n = cfg.dims[0]
    while n > (33 if nd == 3 else 257) and per_node_cycle * float(n) ** nd * est_cycles > seconds_per_solve:
        n = (n - 1) // 2 + 1
    return cfg if n == cfg.dims[0] else I.scaled(cfg, n)


def oracle_solve(cfg, inp):
    """one complete solve by the oracle as it stands (Algorithm H, one thread): cycles until the tolerance, as
    homg_solve does.  -> (seconds, cycles, relative residual)"""
    from oracle import oracle as O
    sched = O.schedule(cfg.schedule, cfg.levels, cfg.max_iters)
    u = inp["u0"].copy()
    t0 = time.perf_counter()
    n0, rel, c = None, 1.0, 0
    while c < cfg.cycles:
        u, _, n = O.homg("H", inp["f"], u, cfg.levels, cfg.omega, sched, 1, k=inp["k"], keep_history=False)
        n0 = n[0] if n0 is None else n0
        c += 1
        rel = n[1] / n0 if n0 > 0 else 0.0
        if cfg.tol > 0 and rel <= cfg.tol:
            break
    return time.perf_counter() - t0, c, rel


def cpu_baseline(cfg, seconds):
    scfg = sample_config(cfg, seconds)
    sec, cyc, rel = oracle_solve(scfg, I.make_inputs(scfg))
    return {"value": scfg.n_interior / sec, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"one complete solve of the same recipe at {'x'.join(map(str, scfg.dims))} ({cyc} cycles to rel. residual "
                      f"{rel:.2e}, {sec:.1f} s); the oracle is single-threaded, untuned test infrastructure (-O2, no SIMD "
                      f"pragmas), cost linear in the nodes",
            "host_cores_available": os.cpu_count()}


def run_reference(args):
    """--impl reference: the oracle (CPU, one thread, as it stands) on a bounded sample of the workload; every step is
    one COMPLETE, fully timed solve.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = I.CONFIGS[args.workload]
    if args.n:
        cfg = I.scaled(cfg, args.n)
    warm = max(1, args.warmup)
    scfg = sample_config(cfg, args.ref_seconds / (args.steps + warm))
    inp = I.make_inputs(scfg)
    for _ in range(warm):
        oracle_solve(scfg, inp)
    t_sum, cyc, rel = 0.0, 0, 1.0
    for _ in range(args.steps):
        sec, cyc, rel = oracle_solve(scfg, inp)
        t_sum += sec
    val = scfg.n_interior * args.steps / t_sum
    sample = (f"every step = one complete solve of the same recipe at {'x'.join(map(str, scfg.dims))} "
              f"({cyc} cycles to rel. residual {rel:.2e}), timed in full")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_sum / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic", "config": workload_config(cfg),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "cycles_to_tol": cyc, "gpu_launches": 0}
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
    own_loop = args.cycle == "mfmg"                       # homg_solve: the MFMG cycle, plain or mixed precision
    s, d = make_solver(cfg, inp, torch, dev, vcycle=(2, 1) if args.cycle == "v" else None,
                       literal=args.cycle == "literal", mixed=args.mixed)
    job = Solve(s, cfg, own_loop)
    if not (own_loop and cfg.tol > 0) and cfg.tol > 0:
        job.find_cstar(d["u0"])
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    sampler = ClockSampler(local)
    stream = torch.cuda.current_stream()

    def sync_all():
        torch.cuda.synchronize()
        replicas.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        flush.zero_()
        job.run(d["u0"])
    sync_all()
    t_a = time.time()
    total_ms, cycles, rel = 0.0, 0, 1.0
    for _ in range(args.steps):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        cycles, rel = job.run(d["u0"])
        e1.record(stream)
        e1.synchronize()
        total_ms += e0.elapsed_time(e1)
    sync_all()
    sampler.mark(t_a, time.time())
    stagnated = cfg.tol > 0 and rel > cfg.tol

    # ---- e2e: host buffers through the C ABI ----
    hf = torch.from_numpy(inp["f"]).pin_memory()
    hu0 = torch.from_numpy(inp["u0"]).pin_memory() if inp["u0"].any() else None     # u0 = 0: the default guess, no upload
    hk = None if inp["k"] is None else torch.from_numpy(inp["k"]).pin_memory()
    hout = torch.empty(cfg.dims, dtype=hf.dtype).pin_memory()

    def step_e2e():
        if hk is not None:
            s.set_coefficient(hk)
        s.set_rhs(hf)
        r = job.run(hu0)
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
    launches_cycle = s.launches_per_cycle()
    prof = {}
    if not args.mixed:                          # (homg_profile_cycles is not available in mixed precision)
        s.set_initial_guess(d["u0"])
        s.profile_cycles(1)                     # warm
        s.set_initial_guess(d["u0"])
        t_c = time.time()
        prof = s.profile_cycles(cycles)
        sampler.mark(t_c, time.time())
    peak, peak_src = peaks()
    comp, comp_total = s.compulsory_bytes_per_cycle()
    rl, shares = roofline_from_profile(prof, peak, peak_src, comp, cycles, cfg.name)
    # kernels of one step: the cycles + the first residual pass of homg_solve (2 kernels) or the closing norm-only
    # pass (2) + the pack of u0 (1; u0 = 0 is a memset)
    launches_step = launches_cycle * cycles + 2 + (1 if d["u0"] is not None else 0)
    bytes_cycle = s.bytes_per_cycle()
    clocks = sampler.stop()

    total_ms, e2e_s = replicas.max_over_ranks([total_ms, e2e_s], device=dev)
    es = 8 if cfg.dtype == "f64" else 4
    nbytes = int(np.prod(cfg.dims)) * es
    ms_cycle = total_ms / args.steps / max(cycles, 1)
    line = {"metric": METRIC, "value": replicas.job_value(cfg.n_interior, args.steps, world, total_ms), "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 (u, f, residual) / f32 (correction cycle)" if args.mixed else cfg.dtype, "data": "synthetic",
            "config": workload_config(cfg, args.cycle),
            "cycles_to_tol": cycles, "cycles_decided_by": "homg_solve (device-side loop)" if own_loop and cfg.tol > 0 else
            ("fixed by the config" if cfg.tol <= 0 else "a first run of the same solve"),
            "rel_residual_reached": float(rel), "stagnated_above_tol": bool(stagnated),
            "ms_per_cycle": ms_cycle, "unknowns_per_s_per_cycle": cfg.n_interior * world / (ms_cycle * 1e-3),
            "cycle_sweep_equiv_gb": bytes_cycle / 1e9, "cycle_hbm_gb": comp_total / 1e9,
            "cycle_hbm_gbs": comp_total / (ms_cycle * 1e-3) / 1e9, "cycle_hbm_frac_of_peak": comp_total / (ms_cycle * 1e-3) / 1e9 / peak,
            "e2e": {"value": cfg.n_interior * n_e2e * world / e2e_s, "unit": UNIT, "ms_per_step": e2e_s / n_e2e * 1e3,
                    "h2d_bytes_per_step": nbytes * (1 + (hk is not None) + (hu0 is not None)), "d2h_bytes_per_step": nbytes + 20},
            "gpu_launches": launches_step * args.steps, "launches_per_cycle": launches_cycle, "roofline": rl, "kernels": shares,
            "clocks": clocks}
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(cfg, args.cpu_seconds)
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
    s, d = make_solver(cfg, inp, torch, dev, vcycle=vcycle, literal=literal)
    job = Solve(s, cfg, False)
    if literal and cfg.n_interior > 3e7:        # (seconds per solve: one capped probe of the cycle count is all it gets)
        import dataclasses
        job.cfg = dataclasses.replace(cfg, cycles=min(cfg.cycles, 12))
    cstar = job.find_cstar(d["u0"]) if cfg.tol > 0 else cfg.cycles
    reps = 1 if literal else 5
    for _ in range(0 if literal else 2):
        job.run(d["u0"])
    ms, fin = 0.0, 1.0
    for _ in range(reps):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        _, fin = job.run(d["u0"])
        e1.record(); e1.synchronize()
        ms += e0.elapsed_time(e1)
    ms /= reps
    out = {"cycles_to_tol": cstar, "ms_per_step": ms, "ms_per_cycle": ms / cstar, "value": cfg.n_interior / (ms * 1e-3),
           "unit": UNIT, "rel_residual_reached": float(fin), "stagnated_above_tol": bool(cfg.tol > 0 and fin > cfg.tol),
           "launches_per_cycle": s.launches_per_cycle()}
    s.destroy()
    return out


def spawn_replicas(args):
    """`python bench.py --gpus N` outside torchrun: launch the N replicas ourselves (one process per GPU)."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    elif a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_replicas(a)
    else:
        run_homg(a)
