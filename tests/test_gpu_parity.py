"""-m gpu: parity of the CUDA path (through the C ABI, via the thin binding) against the oracle.

Bar (BASELINE.json north_star / SURVEY.md 8(d)): after EVERY cycle
    max|u_gpu - u_orc| / max|u_orc| <= 1e-12 (fp64) / 1e-5 (fp32, oracle also in fp32)
and per-cycle residual factors equal to 3 significant digits while above the rounding floor.
Inputs: paper_1108_2045_b200.inputs (seeded, synthetic; shared generator module, no arithmetic).
"""
import numpy as np
import pytest

from paper_1108_2045_b200 import inputs as I

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests")
    return torch


def run_gpu(cfg, inp, ncycles, **kw):
    """Runs ncycles one at a time and returns (list of u after each cycle, norms[ncycles+1])."""
    torch = _torch()
    from paper_1108_2045_b200 import homg
    s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, cfg.dtype, omega=cfg.omega, max_iters=cfg.max_iters,
                    schedule=cfg.schedule, **kw)
    if inp["k"] is not None:
        s.set_coefficient(inp["k"])
    s.set_rhs(inp["f"])
    s.set_initial_guess(inp["u0"])
    us = []
    out = np.empty(cfg.dims, dtype=cfg.np_dtype)
    for _ in range(ncycles):
        s.cycle(1)
        us.append(s.get_solution(out).copy())
    hist = s.residual_history()
    final, rel = s.residual_norm()
    assert len(hist) == ncycles
    norms = np.array(hist + [final])
    assert s.launches_per_cycle() > 0
    sched = s.schedule()
    s.destroy()
    return us, norms, sched


def check_parity(cfg, ncycles, orc, floor=None, **kw):
    inp = I.make_inputs(cfg)
    us, norms, sched = run_gpu(cfg, inp, ncycles, **kw)
    osched = kw.get("sched") or orc.schedule(cfg.schedule, cfg.levels, cfg.max_iters)
    assert (list(sched[0]), list(sched[1])) == (list(osched[0]), list(osched[1]))
    _, hist, onorms = orc.homg("H", inp["f"], inp["u0"], cfg.levels, cfg.omega, osched, ncycles, k=inp["k"])
    tol = TOL[cfg.dtype]
    for c in range(ncycles):
        ref = hist[c].astype(np.float64)
        err = np.max(np.abs(us[c].astype(np.float64) - ref)) / np.max(np.abs(ref))
        assert err <= tol, f"{cfg.name}: cycle {c}: max-norm relative difference {err:.3e} > {tol}"
    # residual factors to 3 significant digits while above the floor
    if floor is None:
        floor = 1e-11 if cfg.dtype == "f64" else 3e-5
    for c in range(1, ncycles + 1):
        if onorms[c] / onorms[0] < floor:
            break
        fg, fo = norms[c] / norms[c - 1], onorms[c] / onorms[c - 1]
        assert abs(fg - fo) <= 5e-4 * abs(fo), (cfg.name, c, fg, fo)       # 3 significant digits (north_star)
    return us, norms


def test_cfg1_full(orc):
    """BASELINE configs[0]: 129^2 fp64, 7 levels, 10 cycles, exactly as stated."""
    cfg = I.CONFIGS["cfg1"]
    us, norms = check_parity(cfg, 10, orc)
    import os
    golden = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "cfg1_norms.txt"), comments="#")
    g = np.atleast_1d(golden).ravel()
    n = min(len(g), len(norms))
    assert np.allclose(norms[:n], g[:n], rtol=1e-9), "GPU norms differ from the oracle-written golden file"


@pytest.mark.parametrize("n", [17, 33, 65])
def test_cfg2_scaled(orc, n):
    check_parity(I.scaled(I.CONFIGS["cfg2"], n), 6, orc)


@pytest.mark.parametrize("n", [65, 257, 513])
def test_cfg3_scaled(orc, n):
    check_parity(I.scaled(I.CONFIGS["cfg3"], n), 5, orc)


@pytest.mark.parametrize("n", [33, 65])
def test_cfg4_scaled(orc, n):
    check_parity(I.scaled(I.CONFIGS["cfg4"], n), 5, orc)


@pytest.mark.parametrize("n", [17, 33, 65])
def test_cfg5_scaled(orc, n):
    check_parity(I.scaled(I.CONFIGS["cfg5"], n), 6, orc)


@pytest.mark.parametrize("kind", [0, 1, 2])
@pytest.mark.parametrize("maxi", [2, 4, 32])
def test_schedules_2d(orc, kind, maxi):
    import dataclasses
    cfg = dataclasses.replace(I.scaled(I.CONFIGS["cfg1"], 65), schedule=kind, max_iters=maxi)
    check_parity(cfg, 3, orc)


@pytest.mark.parametrize("kind", [1, 2])
def test_schedules_3d(orc, kind):
    import dataclasses
    cfg = dataclasses.replace(I.scaled(I.CONFIGS["cfg5"], 33), schedule=kind, max_iters=8)
    check_parity(cfg, 3, orc)


def test_explicit_schedule_with_single_iterations_and_fine_revisits(orc):
    """eta = 1 visits, level 0 visited in mid-schedule, repeated level, multi-level jumps."""
    cfg = I.scaled(I.CONFIGS["cfg1"], 33)
    sched = ([4, 4, 2, 0, 3, 1, 1, 0, 2, 4, 0], [1, 2, 1, 2, 3, 1, 1, 1, 2, 2, 3])
    check_parity(cfg, 3, orc, sched=sched)
    cfg3 = I.scaled(I.CONFIGS["cfg2"], 17)
    sched3 = ([3, 1, 0, 2, 3, 0], [1, 1, 2, 1, 2, 2])
    check_parity(cfg3, 3, orc, sched=sched3)


@pytest.mark.parametrize("fuse_first", ["1", "0"])
def test_explicit_schedule_mid_cycle_fine_visits_on_tiled_levels(orc, monkeypatch, fuse_first):
    """a level-0 visit of eta >= 2 in MID-cycle followed by a move up, on grids where K_visit runs level 0
    (tiled_min_nodes=1): the carried variation of the next visit needs v^{eta-1} of that visit
    (the r01 executor left it unset: ADVICE r1)."""
    monkeypatch.setenv("HOMG_FUSE_FIRST", fuse_first)
    cfg3 = I.scaled(I.CONFIGS["cfg4"], 33)
    sched3 = ([4, 3, 2, 1, 0, 1, 0, 2, 1, 0], [2, 2, 2, 3, 4, 2, 2, 2, 4, 3])
    check_parity(cfg3, 3, orc, sched=sched3, tiled_min_nodes=1)
    cfg64 = I.scaled(I.CONFIGS["cfg2"], 33)
    sched64 = ([4, 2, 0, 1, 0, 3, 0], [2, 4, 6, 2, 5, 1, 4])          # eta > 4 on level 0: chunked K_visit + a trailing sweep
    check_parity(cfg64, 3, orc, sched=sched64, tiled_min_nodes=1)
    cfg2d = I.scaled(I.CONFIGS["cfg3"], 257)
    sched2d = ([7, 6, 3, 1, 0, 1, 0, 2, 0], [2, 2, 4, 4, 4, 2, 3, 2, 2])
    check_parity(cfg2d, 3, orc, sched=sched2d, tiled_min_nodes=1)


def test_ragged_dims_and_fewer_levels(orc):
    """non-square / non-cubic grids, rows that are not a multiple of the 128-B pitch, levels < max."""
    import dataclasses
    base = I.CONFIGS["cfg1"]
    cfg = dataclasses.replace(base, name="cfg1@ragged", dims=(49, 81), levels=4)
    check_parity(cfg, 4, orc)
    base3 = I.CONFIGS["cfg5"]
    cfg3 = dataclasses.replace(base3, name="cfg5@ragged", dims=(17, 41, 25), levels=3)
    check_parity(cfg3, 4, orc)
    cfg4 = dataclasses.replace(I.CONFIGS["cfg4"], name="cfg4@ragged", dims=(9, 13, 37), levels=2)
    check_parity(cfg4, 4, orc)


def test_single_level_and_smallest_grid(orc):
    import dataclasses
    cfg = dataclasses.replace(I.CONFIGS["cfg1"], name="cfg1@1lvl", dims=(9, 9), levels=1)
    check_parity(cfg, 3, orc)
    cfg = dataclasses.replace(I.CONFIGS["cfg2"], name="cfg2@3", dims=(3, 3, 3), levels=1)
    check_parity(cfg, 2, orc)
    cfg = dataclasses.replace(I.CONFIGS["cfg2"], name="cfg2@5", dims=(5, 5, 5), levels=2)
    check_parity(cfg, 3, orc)


def test_graph_and_stream_launch_agree(orc):
    cfg = I.scaled(I.CONFIGS["cfg2"], 33)
    inp = I.make_inputs(cfg)
    a, na, _ = run_gpu(cfg, inp, 3, use_graph=1)
    b, nb, _ = run_gpu(cfg, inp, 3, use_graph=0)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert np.array_equal(na, nb)


def test_device_arrays_and_zero_residual_fixed_point(orc):
    """device-pointer in/out path; f = 0, u0 = 0 stays exactly 0 (pin P1's trivial half on the GPU)."""
    torch = _torch()
    from paper_1108_2045_b200 import homg
    cfg = I.scaled(I.CONFIGS["cfg4"], 33)
    inp = I.make_inputs(cfg)
    s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, cfg.dtype)
    fd = torch.from_numpy(inp["f"]).cuda()
    s.set_rhs(fd)
    s.cycle(3)
    out = torch.empty(cfg.dims, dtype=torch.float32, device="cuda")
    s.get_solution(out)
    host = np.empty(cfg.dims, dtype=np.float32)
    s.get_solution(host)
    assert np.array_equal(out.cpu().numpy(), host)
    s.set_rhs(torch.zeros_like(fd))
    s.set_initial_guess(torch.zeros_like(fd))
    s.cycle(2)
    s.get_solution(host)
    assert not host.any()
    assert s.residual_norm()[0] == 0.0
    s.destroy()


def test_null_initial_guess_is_the_zero_guess(orc):
    """homg_set_initial_guess(NULL) = the default guess u = 0 set on the device (include/homg.h): solving again
    after it reproduces, bit for bit, the solve that started from an uploaded array of zeros."""
    _torch()
    from paper_1108_2045_b200 import homg
    cfg = I.scaled(I.CONFIGS["cfg4"], 65)
    inp = I.make_inputs(cfg)
    assert not inp["u0"].any()
    s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, cfg.dtype, omega=cfg.omega, max_iters=cfg.max_iters)
    s.set_rhs(inp["f"])
    s.set_initial_guess(inp["u0"])
    s.cycle(3)
    a = s.get_solution().copy()
    ha = s.residual_history()
    s.set_initial_guess(None)
    assert s.residual_history() == []
    z = s.get_solution()
    assert not z.any()
    s.cycle(3)
    b = s.get_solution().copy()
    assert np.array_equal(a, b) and s.residual_history() == ha
    s.destroy()


def test_error_paths():
    _torch()
    from paper_1108_2045_b200 import homg
    with pytest.raises(homg.HomgError):
        homg.Solver((130, 129), 7, "poisson5", "f64")
    with pytest.raises(homg.HomgError):
        homg.Solver((129, 129), 7, "poisson7", "f64")
    s = homg.Solver((17, 17), 3, "poisson5", "f64")
    with pytest.raises(homg.HomgError) as ei:
        s.cycle(1)
    assert ei.value.status == homg.HOMG_ESTATE
    s.destroy()
    s = homg.Solver((9, 9, 9), 2, "diffusion7", "f64")
    s.set_rhs(np.ones((9, 9, 9)))
    with pytest.raises(homg.HomgError):
        s.cycle(1)
    s.destroy()


@pytest.mark.parametrize("name,n,chunk", [("cfg2", 33, 0), ("cfg2", 65, 5), ("cfg4", 65, 0), ("cfg4", 129, 16),
                                          ("cfg5", 33, 3), ("cfg5", 65, 0), ("cfg3", 257, 7), ("cfg3", 1025, 0),
                                          ("cfg1", 129, 0)])
def test_tiled_tma_kernels_every_level(orc, name, n, chunk):
    """tiled_min_nodes=1 forces the TMA-tiled kernels on EVERY level (down to 3^d), with ragged
    tiles, several chunks along the marching axis and chunk tails."""
    ncyc = 2 if n >= 129 and name != "cfg1" and name != "cfg3" else 3
    check_parity(I.scaled(I.CONFIGS[name], n), ncyc, orc, tiled_min_nodes=1, march_chunk=chunk)


def test_tiled_matches_generic_bitwise(orc):
    cfg = I.scaled(I.CONFIGS["cfg4"], 65)
    inp = I.make_inputs(cfg)
    a, na, _ = run_gpu(cfg, inp, 3, tiled_min_nodes=1)
    b, nb, _ = run_gpu(cfg, inp, 3, tiled_min_nodes=-1)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("name,n,maxi", [("cfg4", 129, 4), ("cfg2", 65, 3), ("cfg3", 1025, 4), ("cfg4", 65, 8), ("cfg1", 513, 2)])
def test_kvisit_matches_per_sweep_kernels_bitwise(orc, monkeypatch, name, n, maxi):
    """K_visit (all sweeps of a visit in one pass, halo recompute, chunked marching axis) is bit-identical to
    one launch per sweep, at sizes of several tiles with ragged tails, for NS = 2, 3, 4 and chunked visits."""
    import dataclasses
    cfg = dataclasses.replace(I.scaled(I.CONFIGS[name], n), max_iters=maxi)
    inp = I.make_inputs(cfg)
    # (tiled_min_nodes: 65^3 and 513^2 sit below the default threshold of the tiled kernels)
    a, na, _ = run_gpu(cfg, inp, 2, tiled_min_nodes=200000)
    monkeypatch.setenv("HOMG_FUSE_VISIT", "0")
    b, nb, _ = run_gpu(cfg, inp, 2, tiled_min_nodes=200000)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert np.array_equal(na, nb)


def test_variable_coefficient_fused_first_sweep(orc, monkeypatch):
    """k_relax_first for the variable-coefficient stencil (off by default: slower than deliver + sweep on cfg5)."""
    monkeypatch.setenv("HOMG_FUSE_FIRST_VAR", "1")
    check_parity(I.scaled(I.CONFIGS["cfg5"], 65), 3, orc, tiled_min_nodes=200000)
    check_parity(I.scaled(I.CONFIGS["cfg5"], 33), 3, orc, tiled_min_nodes=1, march_chunk=6)


# ---- classic V(eta1, eta2) cycle on the GPU vs the oracle's Algorithm V ----
def check_vcycle(cfg, ncycles, orc, eta=(2, 1), **kw):
    inp = I.make_inputs(cfg)
    us, norms, _ = run_gpu(cfg, inp, ncycles, vcycle=eta, **kw)
    _, hist, onorms = orc.vcycle(inp["f"], inp["u0"], cfg.levels, cfg.omega, eta[0], eta[1], ncycles, k=inp["k"],
                                 keep_history=True)
    tol = TOL[cfg.dtype]
    for c in range(ncycles):
        ref = hist[c].astype(np.float64)
        err = np.max(np.abs(us[c].astype(np.float64) - ref)) / np.max(np.abs(ref))
        assert err <= tol, f"{cfg.name} V{eta}: cycle {c}: max-norm relative difference {err:.3e} > {tol}"
    floor = 1e-11 if cfg.dtype == "f64" else 3e-5
    for c in range(1, ncycles + 1):
        if onorms[c] / onorms[0] < floor:
            break
        fg, fo = norms[c] / norms[c - 1], onorms[c] / onorms[c - 1]
        assert abs(fg - fo) <= 5e-4 * abs(fo), (cfg.name, c, fg, fo)
    return norms


@pytest.mark.parametrize("name,n,eta", [("cfg1", 129, (2, 1)), ("cfg2", 33, (2, 1)), ("cfg2", 65, (1, 1)), ("cfg3", 257, (2, 2)),
                                        ("cfg4", 65, (2, 1)), ("cfg5", 33, (2, 1)), ("cfg4", 33, (0, 1)), ("cfg2", 17, (3, 0)),
                                        ("cfg4", 129, (4, 4))])
def test_vcycle_mode(orc, name, n, eta):
    cfg = I.CONFIGS[name] if I.CONFIGS[name].dims[0] == n else I.scaled(I.CONFIGS[name], n)
    check_vcycle(cfg, 4, orc, eta=eta)


def test_vcycle_tiled_every_level_and_contraction(orc):
    """tiled kernels (K_visit, K_res) on every level; the V(2,1) factor is h-independent and ~ mu^3 (pin P11)."""
    cfg = I.scaled(I.CONFIGS["cfg2"], 65)
    norms = check_vcycle(cfg, 6, orc, eta=(2, 1), tiled_min_nodes=1)
    fac = norms[5] / norms[4]
    assert fac < 0.45, fac


def test_vcycle_needs_one_node_coarsest_level():
    _torch()
    from paper_1108_2045_b200 import homg
    with pytest.raises(homg.HomgError):
        homg.Solver((65, 65, 65), 4, "poisson7", "f64", vcycle=(2, 1))


# ---- paper-literal whole-grid mode (Algorithm L on the GPU) vs the oracle's Algorithm L ----
@pytest.mark.parametrize("name,n,kind,maxi", [("cfg1", 65, 0, 4), ("cfg1", 33, 2, 2), ("cfg2", 17, 0, 4), ("cfg2", 33, 1, 8),
                                              ("cfg4", 33, 0, 4), ("cfg5", 17, 0, 4), ("cfg3", 129, 0, 32)])
def test_literal_mode(orc, name, n, kind, maxi):
    import dataclasses
    cfg = dataclasses.replace(I.scaled(I.CONFIGS[name], n), schedule=kind, max_iters=maxi)
    inp = I.make_inputs(cfg)
    ncyc = 3
    us, norms, sched = run_gpu(cfg, inp, ncyc, literal=True)
    osched = orc.schedule(cfg.schedule, cfg.levels, cfg.max_iters)
    assert (list(sched[0]), list(sched[1])) == (list(osched[0]), list(osched[1]))
    _, hist, onorms = orc.homg("L", inp["f"], inp["u0"], cfg.levels, cfg.omega, osched, ncyc, k=inp["k"])
    tol = TOL[cfg.dtype]
    for c in range(ncyc):
        ref = hist[c].astype(np.float64)
        err = np.max(np.abs(us[c].astype(np.float64) - ref)) / np.max(np.abs(ref))
        assert err <= tol, f"{cfg.name} literal: cycle {c}: {err:.3e} > {tol}"
    assert np.allclose(norms, onorms, rtol=1e-5 if cfg.dtype == "f32" else 1e-10)


def test_literal_and_per_level_forms_agree(orc):
    """Algorithm L (one fine array) and Algorithm H (per-level arrays, the product) give the same u to rounding (pin P7, on the GPU)."""
    cfg = I.scaled(I.CONFIGS["cfg2"], 33)
    inp = I.make_inputs(cfg)
    a, _, _ = run_gpu(cfg, inp, 3, literal=True)
    b, _, _ = run_gpu(cfg, inp, 3)
    for x, y in zip(a, b):
        assert np.max(np.abs(x - y)) <= 1e-12 * np.max(np.abs(y))


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times (graph replay, default
# ---- thresholds): the oracle runs the first cycle(s) of the same solve and EVERY node is compared ----
@pytest.mark.parametrize("name,ncyc", [("cfg2", 14), ("cfg5", 3), ("cfg3", 2), ("cfg4", 2)])
def test_full_size_first_cycles_vs_oracle(orc, name, ncyc):
    """cfg2: the whole solve (14 cycles to 1e-8); cfg3-5: the first cycles.  u is compared after EVERY cycle."""
    cfg = I.CONFIGS[name]
    inp = I.make_inputs(cfg)
    us, norms, sched = run_gpu(cfg, inp, ncyc)
    _, hist, onorms = orc.homg("H", inp["f"], inp["u0"], cfg.levels, cfg.omega, sched, ncyc, k=inp["k"], keep_history=True)
    for c in range(ncyc):
        ref = hist[c]
        err = float(np.max(np.abs(us[c] - ref))) / float(np.max(np.abs(ref)))
        assert err <= TOL[cfg.dtype], f"{name} full size, cycle {c}: {err:.3e}"
    assert np.allclose(norms, onorms, rtol=1e-5 if cfg.dtype == "f32" else 1e-10)
    if name == "cfg2":
        assert onorms[14] <= cfg.tol * onorms[0] < onorms[13]       # 14 cycles is what 1e-8 takes
    # Dirichlet boundary stays exactly 0
    u = us[-1]
    for ax in range(u.ndim):
        assert not np.any(np.take(u, [0, -1], axis=ax))


# ---- homg_solve: the solve stops by itself (a device-side WHILE loop over the cycle) ----
def oracle_cycles_to_tol(orc, cfg, inp, tol, cap):
    sched = orc.schedule(cfg.schedule, cfg.levels, cfg.max_iters)
    _, _, norms = orc.homg("H", inp["f"], inp["u0"], cfg.levels, cfg.omega, sched, cap, k=inp["k"], keep_history=False)
    for c, v in enumerate(norms):
        if v <= tol * norms[0]:
            return c, norms
    return cap, norms


@pytest.mark.parametrize("name,n,tol,kw", [("cfg2", 65, 1e-8, {}), ("cfg5", 33, 1e-8, {}), ("cfg4", 65, 1e-4, {"tiled_min_nodes": 200000}),
                                           ("cfg3", 513, 1e-3, {"tiled_min_nodes": 200000}), ("cfg1", 129, 1e-6, {}),
                                           ("cfg2", 33, 1e-8, {"tiled_min_nodes": 1})])
def test_solve_stops_by_itself(orc, name, n, tol, kw):
    _torch()
    from paper_1108_2045_b200 import homg
    cfg = I.CONFIGS[name] if I.CONFIGS[name].dims[0] == n else I.scaled(I.CONFIGS[name], n)
    inp = I.make_inputs(cfg)
    cap = 40
    want, onorms = oracle_cycles_to_tol(orc, cfg, inp, tol, cap)
    assert 2 <= want < cap
    def mk():
        s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, cfg.dtype, omega=cfg.omega, max_iters=cfg.max_iters, **kw)
        if inp["k"] is not None:
            s.set_coefficient(inp["k"])
        s.set_rhs(inp["f"])
        s.set_initial_guess(inp["u0"])
        return s
    s = mk()
    done, rel = s.solve(tol, cap)
    assert done == want, (done, want)                                   # the oracle's count
    u = s.get_solution().copy()
    hist = s.residual_history()
    assert len(hist) == done
    assert np.allclose(hist, onorms[:done], rtol=1e-5 if cfg.dtype == "f32" else 1e-10)
    final, rel2 = s.residual_norm()
    assert abs(rel - rel2) <= 1e-12 * rel2 and rel <= tol
    assert abs(final - onorms[done]) <= (1e-5 if cfg.dtype == "f32" else 1e-10) * onorms[done]
    # the same cycles issued one by one give the same u, bit for bit
    r = mk()
    r.cycle(done)
    assert np.array_equal(r.get_solution(), u)
    assert r.residual_history() == hist
    # the cap stops the loop; solving on continues from where it is; homg_cycle after homg_solve appends
    t = mk()
    d1, rel1 = t.solve(tol, 2)
    assert d1 == 2 and rel1 > tol
    d2, _ = t.solve(tol, cap)
    assert d1 + d2 == want and np.array_equal(t.get_solution(), u)
    d3, _ = t.solve(tol, cap)
    assert d3 == 0                                                      # already converged: no cycle runs
    t.cycle(1)
    assert len(t.residual_history()) == want + 1
    r.cycle(1)
    assert np.array_equal(t.get_solution(), r.get_solution())
    assert t.residual_history() == r.residual_history()
    for x in (s, r, t):
        x.destroy()


def test_solve_argument_checks():
    _torch()
    from paper_1108_2045_b200 import homg
    s = homg.Solver((17, 17), 3, "poisson5", "f64")
    with pytest.raises(homg.HomgError) as ei:
        s.solve(1e-8, 10)
    assert ei.value.status == homg.HOMG_ESTATE
    s.set_rhs(np.ones((17, 17)))
    with pytest.raises(homg.HomgError):
        s.solve(-1.0, 10)
    with pytest.raises(homg.HomgError):
        s.solve(1e-8, 5000)                                             # history_cap (4096) too small
    assert s.solve(1e-8, 0)[0] == 0
    s.destroy()
    v = homg.Solver((17, 17), 4, "poisson5", "f64", vcycle=(2, 1))
    v.set_rhs(np.ones((17, 17)))
    with pytest.raises(homg.HomgError) as ei:
        v.solve(1e-8, 10)
    assert ei.value.status == homg.HOMG_ESTATE
    v.destroy()


# ---- mixed-precision outer loop vs the oracle's mixed loop: fp64 u, f, r; fp32 correction cycle ----
@pytest.mark.parametrize("name,n", [("cfg2", 33), ("cfg2", 65), ("cfg1", 129), ("cfg5", 33), ("cfg5", 65)])
def test_mixed_precision_mode(orc, name, n):
    cfg = I.CONFIGS[name] if I.CONFIGS[name].dims[0] == n else I.scaled(I.CONFIGS[name], n)
    assert cfg.dtype == "f64"
    inp = I.make_inputs(cfg)
    ncyc = 8
    us, norms, sched = run_gpu(cfg, inp, ncyc, mixed=True)
    _, hist, onorms = orc.homg_mixed(inp["f"], inp["u0"], cfg.levels, cfg.omega, sched, ncyc, k=inp["k"])
    for c in range(ncyc):
        err = np.max(np.abs(us[c] - hist[c])) / np.max(np.abs(hist[c]))
        assert err <= 1e-12, f"{cfg.name} mixed: cycle {c}: {err:.3e}"
    assert np.allclose(norms, onorms, rtol=1e-9)


def test_mixed_precision_keeps_contracting_below_the_fp32_floor(orc):
    """the fp64 outer residual keeps contracting where the pure fp32 solve stalls at its rounding floor."""
    import dataclasses
    cfg = I.scaled(I.CONFIGS["cfg2"], 65)
    inp = I.make_inputs(cfg)
    _, norms, _ = run_gpu(cfg, inp, 30, mixed=True)
    assert norms[-1] <= 1e-12 * norms[0]
    cfg32 = dataclasses.replace(cfg, dtype="f32")
    inp32 = {k: (None if v is None else v.astype(np.float32)) for k, v in inp.items()}
    _, n32, _ = run_gpu(cfg32, inp32, 30)
    assert norms[-1] / norms[0] < 1e-3 * n32[-1] / n32[0]


def test_mixed_precision_argument_checks():
    _torch()
    from paper_1108_2045_b200 import homg
    with pytest.raises(homg.HomgError):
        homg.Solver((33, 33, 33), 5, "poisson7", "f64", mixed=True, vcycle=(2, 1))


# ---- compute-sanitizer is closed on this GPU pool (profiles/r02_sanitizer.md): the checks that remain ours ----
@pytest.mark.parametrize("name,n,kw", [("cfg4", 65, {"tiled_min_nodes": 1}), ("cfg2", 33, {"tiled_min_nodes": 1}),
                                       ("cfg3", 513, {"tiled_min_nodes": 1}), ("cfg5", 33, {"tiled_min_nodes": 1}),
                                       ("cfg1", 129, {}), ("cfg4", 33, {"tiled_min_nodes": 1, "vcycle": True}),
                                       ("cfg2", 33, {"tiled_min_nodes": 1, "mixed": True})])
def test_no_write_outside_the_workspace(name, n, kw):
    """the solver lives in a caller-owned workspace: 4 MiB of canaries on either side of it stay untouched by every
    kernel family (ragged tiles, halo packs, TMA boxes, 16-byte row tails), and every array inside stays finite."""
    import ctypes as C
    torch = _torch()
    from paper_1108_2045_b200 import homg
    cfg = I.CONFIGS[name] if I.CONFIGS[name].dims[0] == n else I.scaled(I.CONFIGS[name], n)
    inp = I.make_inputs(cfg)
    mixed = kw.pop("mixed", False)
    vc = kw.pop("vcycle", False)
    L = homg.lib()
    dims = homg._dims(cfg.dims)
    dt = "f64" if mixed else cfg.dtype
    if mixed:
        inp = {k: (None if v is None else v.astype(np.float64)) for k, v in inp.items()}
        need = L.homg_workspace_bytes_mixed(len(cfg.dims), dims, cfg.levels, homg.STENCILS[cfg.stencil])
    else:
        need = L.homg_workspace_bytes(len(cfg.dims), dims, cfg.levels, homg.STENCILS[cfg.stencil], homg.DTYPES[dt])
    pad = 4 << 20
    buf = torch.full((need + 2 * pad,), 0xA5, dtype=torch.uint8, device="cuda")
    o = homg.HomgOptions()
    L.homg_default_options(C.byref(o))
    o.omega, o.max_iters, o.tiled_min_nodes = cfg.omega, cfg.max_iters, int(kw.get("tiled_min_nodes", 0))
    o.cuda_stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if vc:
        o.cycle, o.v_eta1, o.v_eta2 = 1, 2, 1
    if mixed:
        o.mixed = 1
    h = C.c_void_p(None)
    assert (buf.data_ptr() + pad) % 256 == 0
    rc = L.homg_create(C.byref(h), len(cfg.dims), dims, cfg.levels, homg.STENCILS[cfg.stencil], homg.DTYPES[dt],
                       C.c_void_p(buf.data_ptr() + pad), need, C.byref(o))
    assert rc == 0, L.homg_last_error(None)
    dev = {k: (None if v is None else torch.from_numpy(v).cuda()) for k, v in inp.items()}
    if dev["k"] is not None:
        assert L.homg_set_coefficient(h, C.c_void_p(dev["k"].data_ptr()), 1) == 0
    assert L.homg_set_rhs(h, C.c_void_p(dev["f"].data_ptr()), 1) == 0
    assert L.homg_set_initial_guess(h, C.c_void_p(dev["u0"].data_ptr()), 1) == 0
    assert L.homg_cycle(h, 3) == 0
    if not vc and not mixed:
        nd, rr = C.c_int(0), C.c_double(0)
        assert L.homg_solve(h, 1e-30, 2, C.byref(nd), C.byref(rr)) == 0 and nd.value == 2
    a, r = C.c_double(0), C.c_double(0)
    assert L.homg_residual_norm(h, C.byref(a), C.byref(r)) == 0 and np.isfinite(a.value)
    out = torch.empty(cfg.dims, dtype=dev["f"].dtype, device="cuda")
    assert L.homg_get_solution(h, C.c_void_p(out.data_ptr()), 1) == 0
    torch.cuda.synchronize()
    assert bool((buf[:pad] == 0xA5).all()) and bool((buf[pad + need:] == 0xA5).all()), "a kernel wrote outside the workspace"
    assert bool(torch.isfinite(out).all())
    L.homg_destroy(h)


def test_a_cycle_is_one_graph_of_kernels_and_memsets_only():
    """"no host transfers inside a solve" (north_star): homg_cycle(n) = n replays of one CUDA graph, homg_solve = one
    launch of a graph with a device-side WHILE node; neither graph holds a memcpy or host node."""
    _torch()
    from paper_1108_2045_b200 import homg
    for name, n, kw in (("cfg4", 65, {"tiled_min_nodes": 200000}), ("cfg1", 129, {}), ("cfg5", 33, {})):
        cfg = I.CONFIGS[name] if I.CONFIGS[name].dims[0] == n else I.scaled(I.CONFIGS[name], n)
        inp = I.make_inputs(cfg)
        s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, cfg.dtype, omega=cfg.omega, max_iters=cfg.max_iters, **kw)
        if inp["k"] is not None:
            s.set_coefficient(inp["k"])
        s.set_rhs(inp["f"])
        s.cycle(1)
        s.solve(1e-3, 5)
        for which in (0, 1):
            c = s.graph_nodes(which)
            assert c["kernel"] == s.launches_per_cycle() + (2 if which == 1 else 0), (name, which, c)
            assert c["memcpy"] == 0 and c["other"] == 0, (name, which, c)
            assert c["conditional"] == which
        s.destroy()


# ---- PAPER.md section 3: power-of-two grids (HOMG_POISSON5_POW2, homg_pow2.cuh) vs the oracle's Algorithm P ----
@pytest.mark.parametrize("N,dtype,levels,kind,maxi,fkind", [(16, "f64", 4, 0, 4, "sine"), (32, "f64", 5, 0, 2, "noise"),
                                                           (64, "f64", 6, 1, 4, "noise"), (64, "f64", 4, 2, 8, "sine"),
                                                           (128, "f32", 7, 0, 4, "noise"), (256, "f64", 8, 0, 4, "noise"),
                                                           (1024, "f64", 10, 0, 4, "noise"), (512, "f32", 9, 0, 32, "sine")])
def test_pow2_grids(orc, N, dtype, levels, kind, maxi, fkind):
    _torch()
    from paper_1108_2045_b200 import homg
    npdt = np.float64 if dtype == "f64" else np.float32
    f = I.sine_rhs((N, N)) + I.uniform_field((N, N), 11, -1e-3, 1e-3) if fkind == "sine" else I.normal_field((N, N), 12)
    f = np.ascontiguousarray(f, dtype=npdt)
    u0 = np.ascontiguousarray(I.uniform_field((N, N), 13, -1.0, 1.0) if fkind == "noise" else np.zeros((N, N)), dtype=npdt)
    ncyc = 3
    s = homg.Solver((N, N), levels, "poisson5_pow2", dtype, omega=0.8, max_iters=maxi, schedule=kind)
    s.set_rhs(f)
    s.set_initial_guess(u0)
    us = []
    for _ in range(ncyc):
        s.cycle(1)
        us.append(s.get_solution().copy())
    norms = np.array(s.residual_history() + [s.residual_norm()[0]])
    sched = s.schedule()
    osched = orc.schedule(kind, levels, maxi)
    assert (list(sched[0]), list(sched[1])) == (list(osched[0]), list(osched[1]))
    s.destroy()
    _, hist, onorms = orc.homg_p2(f, u0, levels, 0.8, osched, ncyc)
    for c in range(ncyc):
        ref = hist[c].astype(np.float64)
        err = np.max(np.abs(us[c].astype(np.float64) - ref)) / np.max(np.abs(ref))
        assert err <= TOL[dtype], f"pow2 N={N}: cycle {c}: {err:.3e}"
    assert np.allclose(norms, onorms, rtol=1e-5 if dtype == "f32" else 1e-10)
    for ax in range(2):
        assert not np.any(np.take(us[-1], [0, -1], axis=ax))


def test_pow2_contraction_and_argument_checks():
    """PAPER.md section 3 on the GPU, reading R19: with the default MaxI of this stencil (32, the paper's L121) a random
    error contracts by < 0.1 per cycle on every grid; with MaxI = 4 the factor grows with N (the oracle pin P12h) and the
    iteration diverges at 2048^2 — the documented limitation of the reading, checked here so that it stays documented."""
    _torch()
    from paper_1108_2045_b200 import homg
    def factor(N, maxi):
        k = int(np.log2(N))
        s = homg.Solver((N, N), k, "poisson5_pow2", "f64", omega=0.8, max_iters=maxi)
        s.set_rhs(np.zeros((N, N)))
        s.set_initial_guess(np.ascontiguousarray(I.uniform_field((N, N), 7, -1.0, 1.0)))
        s.cycle(10)
        h = s.residual_history() + [s.residual_norm()[0]]
        assert s.schedule()[1][-1] == (32 if maxi <= 0 else min(maxi, 2 ** k))
        s.destroy()
        return h[10] / h[9]
    for N in (64, 256, 1024, 2048):
        assert factor(N, 0) < 0.1
    f4 = [factor(N, 4) for N in (64, 256, 1024, 2048)]
    assert f4 == sorted(f4) and f4[0] < 0.26 and 0.7 < f4[2] < 0.95 and f4[3] > 1.0, f4
    with pytest.raises(homg.HomgError):
        homg.Solver((64, 64), 7, "poisson5_pow2", "f64")            # l = 64 > N/2
    with pytest.raises(homg.HomgError):
        homg.Solver((65, 65), 5, "poisson5_pow2", "f64")
    with pytest.raises(homg.HomgError):
        homg.Solver((64, 32), 4, "poisson5_pow2", "f64")
    with pytest.raises(homg.HomgError):
        homg.Solver((64, 64), 5, "poisson5_pow2", "f64", vcycle=(2, 1))


def test_brick_and_pack_level_change_kernels_agree_bitwise(orc, monkeypatch):
    """homg_bricks.cuh (2 x 2 fine rows per thread, used on fine levels of >= 10^6 nodes) against homg_moves.cuh (one
    pack per thread): same arithmetic term by term, hence the same bits — 3-D fp32 / fp64, 2-D, and the V cycle."""
    import dataclasses
    for name, n, kw in (("cfg4", 129, {}), ("cfg5", 129, {}), ("cfg3", 2049, {}), ("cfg4", 129, {"vcycle": (2, 1)})):
        cfg = dataclasses.replace(I.scaled(I.CONFIGS[name], n))
        inp = I.make_inputs(cfg)
        monkeypatch.setenv("HOMG_BRICKS", "1")
        a, na, _ = run_gpu(cfg, inp, 2, **kw)
        monkeypatch.setenv("HOMG_BRICKS", "0")
        b, nb, _ = run_gpu(cfg, inp, 2, **kw)
        for x, y in zip(a, b):
            assert np.array_equal(x, y), (name, n, kw)
        assert np.array_equal(na, nb)


@pytest.mark.parametrize("n,kw", [(65, {"tiled_min_nodes": 200000}), (129, {}), (129, {"march_chunk": 20}), (33, {"tiled_min_nodes": 1})])
def test_variable_coefficient_kvisit_vs_per_sweep_kernels_and_oracle(orc, monkeypatch, n, kw):
    """K_visit for the variable-coefficient stencil (k_visit3<VAR>: interpolate+correct + 2 sweeps, then
    2 sweeps + u += e; the face arrays and omega/D staged by TMA once per pass).  It multiplies by the precomputed
    RN(omega/D) where the per-sweep kernels and the oracle divide (R14): agreement to rounding, not bit for bit
    — <= 1e-13 against the per-sweep path, <= 1e-12 against the oracle after every cycle (cfg5's recipe)."""
    cfg = I.scaled(I.CONFIGS["cfg5"], n)
    inp = I.make_inputs(cfg)
    ncyc = 6
    monkeypatch.setenv("HOMG_VISIT_VAR", "1")
    a, na, _ = run_gpu(cfg, inp, ncyc, **kw)
    monkeypatch.setenv("HOMG_VISIT_VAR", "0")
    b, nb, _ = run_gpu(cfg, inp, ncyc, **kw)
    worst = max(float(np.max(np.abs(x - y)) / np.max(np.abs(y))) for x, y in zip(a, b))
    assert 0 < worst <= 1e-13, worst                 # (> 0: the fused form really ran)
    assert np.allclose(na, nb, rtol=1e-9)
    monkeypatch.setenv("HOMG_VISIT_VAR", "1")
    check_parity(cfg, ncyc, orc, **kw)
    if n == 65:                                     # the mixed-precision loop keeps the bit-exact per-sweep kernels
        us, norms, sched = run_gpu(cfg, inp, 4, mixed=True, **kw)
        _, hist, onorms = orc.homg_mixed(inp["f"], inp["u0"], cfg.levels, cfg.omega, sched, 4, k=inp["k"])
        for c in range(4):
            assert np.max(np.abs(us[c] - hist[c])) <= 1e-12 * np.max(np.abs(hist[c]))


def test_3d_kvisit_forms_agree_bitwise(orc, monkeypatch):
    """k_visit3 (homg_visit3.cuh, the default) and the 3-D form of k_visit (homg_visit.cuh, HOMG_VISIT3=0: the fallback)
    run the same visits with different tiles, pipelines and instruction selection (packed pairs, multiplier instead
    of select): the same bits, level 0 and the bookkeeping form of levels >= 1."""
    for name, n in (("cfg4", 129), ("cfg2", 65)):
        cfg = I.scaled(I.CONFIGS[name], n)
        inp = I.make_inputs(cfg)
        out = {}
        for v in ("2", "1", "0"):
            monkeypatch.setenv("HOMG_VISIT3", v)
            out[v] = run_gpu(cfg, inp, 2, tiled_min_nodes=200000)
        for v in ("1", "0"):
            for x, y in zip(out["2"][0], out[v][0]):
                assert np.array_equal(x, y), (name, v)
            assert np.array_equal(out["2"][1], out[v][1])


@pytest.mark.parametrize("name,n,tol", [("cfg2", 65, 1e-10), ("cfg5", 33, 1e-9), ("cfg1", 129, 1e-8)])
def test_solve_stops_by_itself_in_mixed_precision(orc, name, n, tol):
    """homg_solve around the mixed-precision outer loop (fp64 residual and norm at the end of every cycle set the loop
    condition): the oracle's mixed loop needs the same number of cycles, and the cycles issued one by one give the
    same u bit for bit."""
    _torch()
    from paper_1108_2045_b200 import homg
    cfg = I.CONFIGS[name] if I.CONFIGS[name].dims[0] == n else I.scaled(I.CONFIGS[name], n)
    inp = I.make_inputs(cfg)
    cap = 40
    def mk():
        s = homg.Solver(cfg.dims, cfg.levels, cfg.stencil, "f64", omega=cfg.omega, max_iters=cfg.max_iters, mixed=True)
        if inp["k"] is not None:
            s.set_coefficient(inp["k"])
        s.set_rhs(inp["f"])
        s.set_initial_guess(inp["u0"])
        return s
    s = mk()
    done, rel = s.solve(tol, cap)
    sched = s.schedule()
    _, _, onorms = orc.homg_mixed(inp["f"], inp["u0"], cfg.levels, cfg.omega, sched, cap, k=inp["k"], keep_history=False)
    want = next(c for c, v in enumerate(onorms) if v <= tol * onorms[0])
    assert done == want and 2 <= want < cap and rel <= tol
    u = s.get_solution().copy()
    hist = s.residual_history()
    assert len(hist) == done and np.allclose(hist, onorms[:done], rtol=1e-9)
    r = mk()
    r.cycle(done)
    assert np.array_equal(r.get_solution(), u) and r.residual_history() == hist
    d2, _ = s.solve(tol, cap)
    assert d2 == 0
    s.destroy(); r.destroy()
