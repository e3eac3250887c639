"""Pins for the oracle's whole HOMG cycle and its V-cycle.

  P1  fixed point = dense LU solve (Eq. 1)
  P6  the first iterations of a cycle: spike, then pyramid
  P7  literal single-array algorithm == per-level algorithm; linearity
  P8  the paper's printed L1 errors after one MFMG cycle (Eq. 5-7) — loose
  P9  O(h^2) discretisation error against manufactured solutions
  P10 cost per cycle linear in node count
  P11 classic V-cycle: converges to the LU solution, h-independent factor
"""
import numpy as np
import pytest

from paper_1108_2045_b200 import inputs as I


def test_schedule_tables(orc):
    # two iterations on the coarsest level, doubling per finer level up to MaxI
    lv, it = orc.schedule(0, 7, 4)
    assert lv == [6, 5, 6, 4, 5, 3, 4, 2, 3, 1, 2, 0]
    assert it == [2, 4, 2, 4, 4, 4, 4, 4, 4, 4, 4, 4]
    lv, it = orc.schedule(0, 7, 32)
    assert [i for l, i in zip(lv, it) if l == 6] == [2, 2]
    assert dict(zip(lv, it)) == {6: 2, 5: 4, 4: 8, 3: 16, 2: 32, 1: 32, 0: 32}
    lv, it = orc.schedule(0, 7, 2)
    assert set(it) == {2} and sum(it) == 24
    lv, it = orc.schedule(2, 3, 4)
    assert lv == [2, 2, 1, 2, 1, 0]
    lv, it = orc.schedule(1, 4, 4)
    assert lv == [3, 2, 3, 2, 1, 2, 1, 0]
    assert orc.schedule(0, 1, 4) == ([0], [2])


@pytest.mark.parametrize("shape,levels,omega,var", [
    ((9, 9), 3, 0.8, False), ((17, 17), 4, 0.8, False), ((9, 17), 3, 0.8, False),
    ((9, 9, 9), 3, 6 / 7, False), ((9, 9), 3, 0.8, True), ((9, 9, 9), 3, 6 / 7, True),
    ((17, 17), 2, 0.8, False)])
def test_P1_fixed_point_is_dense_LU(orc, shape, levels, omega, var):
    rng = np.random.default_rng(11)
    f = rng.standard_normal(shape)
    k = np.exp(rng.uniform(-1, 1, shape)) if var else None
    ud = orc.dense_solve(f, k=k)
    # independent check of the LU itself with numpy on the assembled matrix
    A = orc.assemble(shape, k=k)
    inner = tuple(slice(1, -1) for _ in shape)
    un = np.linalg.solve(A, f[inner].ravel()).reshape([n - 2 for n in shape])
    assert np.allclose(ud[inner], un, rtol=0, atol=1e-12 * np.abs(un).max())
    for alg in ("H", "L"):
        u, _, norms = orc.homg(alg, f, np.zeros(shape), levels, omega, orc.schedule(0, levels, 4), 120 if levels > 2 else 600, k=k,
                               keep_history=False)
        assert np.abs(u - ud).max() <= 1e-12 * np.abs(ud).max()
        assert norms[-1] < 1e-11 * norms[0]
    # started AT the fixed point the cycle returns a zero correction (up to rounding of r)
    u2, _, _ = orc.homg("H", f, ud, levels, omega, orc.schedule(0, levels, 4), 1, k=k, keep_history=False)
    assert np.abs(u2 - ud).max() <= 1e-13 * np.abs(ud).max()


@pytest.mark.parametrize("n,d,omega", [(17, 2, 0.8), (17, 2, 1.0), (9, 3, 6 / 7), (33, 2, 0.8)])
def test_P6_spike_then_pyramid(orc, n, d, omega):
    """iteration 1 = spike at the middle node; iteration 2 = relaxation of the
    middle node plus the delayed interpolation of iteration 1 forming a pyramid."""
    shape = (n,) * d
    levels = int(np.log2(n - 1))
    rng = np.random.default_rng(2)
    f = np.zeros(shape)
    f[tuple(slice(1, -1) for _ in shape)] = rng.standard_normal([n - 2] * d)
    sched = orc.schedule(0, levels, 2)
    # g_M(centre) by repeated full weighting, done here with numpy slicing (independent of oracle)
    g = f.copy()
    for _ in range(levels - 1):
        m = g.shape[0]
        acc = np.zeros([(m - 1) // 2 + 1] * d)
        import itertools
        for off in itertools.product((-1, 0, 1), repeat=d):
            w = 2.0 ** (-d - sum(abs(o) for o in off))
            sl = tuple(slice(2 + o, m - 2 + o + 1, 2) for o in off)
            acc[tuple(slice(1, -1) for _ in range(d))] += w * g[sl]
        g = acc
    assert g.shape == (3,) * d
    gc = g[(1,) * d]
    hM = 0.5
    s = omega * hM ** 2 * gc / (2 * d)
    c = (n // 2,) * d
    cur1 = orc.homg_L_partial(f, np.zeros(shape), levels, omega, sched, 1)
    assert abs(cur1[c] - s) <= 1e-14 * abs(s)
    cur1[c] = 0
    assert np.all(cur1 == 0)
    cur2 = orc.homg_L_partial(f, np.zeros(shape), levels, omega, sched, 2)
    assert abs(cur2[c] - omega * (2 - omega) * hM ** 2 * gc / (2 * d)) <= 1e-14 * abs(s)
    x = np.arange(n) / (n - 1)
    hat = 1 - np.abs(2 * x - 1)
    pyr = s
    for a in range(d):
        sh = [1] * d
        sh[a] = n
        pyr = pyr * hat.reshape(sh)
    cur2[c] = pyr[c]
    assert np.allclose(cur2, pyr, rtol=0, atol=1e-14 * abs(s))
    if omega == 1.0:   # "the relaxations have stalled"
        cur2b = orc.homg_L_partial(f, np.zeros(shape), levels, omega, sched, 2)
        assert abs(cur2b[c] - s) <= 1e-14 * abs(s)
    # iteration 3 works on the next finer level: its 3^d-minus-centre lattice nodes now relax
    cur3 = orc.homg_L_partial(f, np.zeros(shape), levels, omega, sched, 3)
    q = (n // 4,) * d
    assert abs(cur3[q] - pyr[q]) > 1e-6 * abs(s)


@pytest.mark.parametrize("shape,levels,omega", [((17, 17), 4, 0.8), ((33, 33), 5, 0.8), ((9, 9, 9), 3, 6 / 7),
                                                ((17, 17, 17), 4, 6 / 7), ((17, 33), 4, 0.8), ((33, 33), 3, 0.8)])
def test_P7_literal_equals_hierarchical(orc, shape, levels, omega):
    rng = np.random.default_rng(0)
    f = rng.standard_normal(shape)
    u0 = rng.standard_normal(shape)
    for a in range(len(shape)):
        sl = [slice(None)] * len(shape)
        for e in (0, -1):
            sl[a] = e
            u0[tuple(sl)] = 0
    for kind in (0, 1, 2):
        for mi in (2, 4, 32):
            s = orc.schedule(kind, levels, mi)
            uL, _, nL = orc.homg("L", f, u0, levels, omega, s, 2, keep_history=False)
            uH, _, nH = orc.homg("H", f, u0, levels, omega, s, 2, keep_history=False)
            assert np.abs(uL - uH).max() <= 1e-13 * np.abs(uL).max(), (kind, mi)
            assert np.allclose(nL, nH, rtol=1e-12)


def test_P7_literal_equals_hierarchical_variable_k_and_odd_schedule(orc):
    rng = np.random.default_rng(4)
    shape = (17, 17, 9)
    f = rng.standard_normal(shape)
    k = np.exp(rng.uniform(-1, 1, shape))
    for s in [orc.schedule(0, 3, 4), ([2, 1, 2, 0, 1, 0], [1, 3, 2, 1, 1, 5]), ([0, 2, 1, 0], [3, 2, 1, 2])]:
        uL, _, _ = orc.homg("L", f, np.zeros(shape), 3, 6 / 7, s, 2, k=k, keep_history=False)
        uH, _, _ = orc.homg("H", f, np.zeros(shape), 3, 6 / 7, s, 2, k=k, keep_history=False)
        assert np.abs(uL - uH).max() <= 1e-13 * np.abs(uL).max()


def test_P7_cycle_is_linear_and_contracts_like_its_matrix(orc):
    shape, levels, omega = (9, 9), 3, 0.8
    sched = orc.schedule(0, levels, 4)
    rng = np.random.default_rng(6)
    z = np.zeros(shape)
    f1, f2 = rng.standard_normal(shape), rng.standard_normal(shape)
    e1 = orc.homg("H", f1, z, levels, omega, sched, 1, keep_history=False)[0]
    e2 = orc.homg("H", f2, z, levels, omega, sched, 1, keep_history=False)[0]
    e12 = orc.homg("H", 2 * f1 - 3 * f2, z, levels, omega, sched, 1, keep_history=False)[0]
    assert np.allclose(e12, 2 * e1 - 3 * e2, atol=1e-13 * np.abs(e12).max())
    # assemble B (e = B r) column by column; asymptotic factor = rho(I - B A)
    inner = (slice(1, -1),) * 2
    N = 49
    B = np.zeros((N, N))
    for j in range(N):
        r = np.zeros(N)
        r[j] = 1
        f = np.zeros(shape)
        f[inner] = r.reshape(7, 7)
        B[:, j] = orc.homg("H", f, z, levels, omega, sched, 1, keep_history=False)[0][inner].ravel()
    A = orc.assemble(shape)
    rho = np.abs(np.linalg.eigvals(np.eye(N) - B @ A)).max()
    assert 0.05 < rho < 0.5
    _, _, norms = orc.homg("H", f1, z, levels, omega, sched, 30, keep_history=False)
    fac = norms[1:] / norms[:-1]
    ok = norms[1:] > 1e-10 * norms[0]
    assert abs(fac[ok][-1] - rho) < 0.02 * rho + 5e-3


def test_P8_paper_L1_errors_after_one_cycle(orc):
    """'MaxI = 4 reaches an error of 5% and MaxI = 32 reaches an error of 1.6%';
    'the same convergence path for different resolutions'.  Loose: the paper's omega is unknown."""
    res = {}
    for n in (65, 129):
        shape = (n, n)
        f, uex = I.paper_polynomial(shape)
        levels = int(np.log2(n - 1))
        for mi in (4, 32):
            u, _, _ = orc.homg("H", f, np.zeros(shape), levels, 0.8, orc.schedule(0, levels, mi), 1,
                               keep_history=False)
            res[(n, mi)] = np.abs(u - uex).sum() / np.abs(uex).sum()     # Eq. 7
    for n in (65, 129):
        assert 0.035 < res[(n, 4)] < 0.065, res
        assert 0.010 < res[(n, 32)] < 0.022, res
    assert abs(res[(65, 4)] - res[(129, 4)]) < 0.01
    # literal algorithm gives the same number
    f, uex = I.paper_polynomial((65, 65))
    uL, _, _ = orc.homg("L", f, np.zeros((65, 65)), 6, 0.8, orc.schedule(0, 6, 4), 1, keep_history=False)
    assert abs(np.abs(uL - uex).sum() / np.abs(uex).sum() - res[(65, 4)]) < 1e-12


def test_P9_second_order_convergence(orc):
    errs = []
    for n in (17, 33, 65):
        shape = (n, n)
        f, uex = I.paper_polynomial(shape)
        levels = int(np.log2(n - 1))
        u, _, norms = orc.homg("H", f, np.zeros(shape), levels, 0.8, orc.schedule(0, levels, 4), 40,
                               keep_history=False)
        assert norms[-1] < 1e-10 * norms[0]
        errs.append(np.abs(u - uex).max())
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.7 < errs[1] / errs[2] < 4.3
    errs = []
    for n in (9, 17, 33):
        shape = (n,) * 3
        f = I.sine_rhs(shape)
        x = np.arange(n) / (n - 1)
        s = np.sin(np.pi * x)
        uex = s[:, None, None] * s[None, :, None] * s[None, None, :]
        levels = int(np.log2(n - 1))
        u, _, _ = orc.homg("H", f, np.zeros(shape), levels, 6 / 7, orc.schedule(0, levels, 4), 40,
                           keep_history=False)
        errs.append(np.abs(u - uex).max())
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.7 < errs[1] / errs[2] < 4.3


def test_P10_cost_linear_in_nodes(orc):
    per_node = []
    for n in (33, 65, 129):
        shape = (n, n)
        levels = int(np.log2(n - 1))
        f = np.ones(shape)
        orc.counters(reset=True)
        orc.homg("H", f, np.zeros(shape), levels, 0.8, orc.schedule(0, levels, 4), 1, keep_history=False)
        relax, moves = orc.counters(reset=True)
        per_node.append((relax / n ** 2, moves / n ** 2))
    r = [p[0] for p in per_node]
    # limit: 4 (level 0) + 4/4 (level 1, one visit) + 8 * sum_{m>=2} 4^-m = 5.667; interior-only counts approach it from below
    assert r[0] < r[1] < r[2] < 4 + 1 + 8 / 12 and r[2] > 5.3 and (r[2] - r[1]) < 0.6 * (r[1] - r[0])
    mv = [p[1] for p in per_node]
    assert max(mv) < 4.5 and max(mv) - min(mv) < 0.6          # moves per fine node: bounded, size independent
    # the literal algorithm costs one whole-grid pass per iteration (1 WU each)
    shape = (33, 33)
    orc.counters(reset=True)
    lv, it = orc.schedule(0, 5, 4)
    orc.homg("L", np.ones(shape), np.zeros(shape), 5, 0.8, (lv, it), 1, keep_history=False)
    relax, moves = orc.counters(reset=True)
    assert relax + moves <= sum(it) * 33 * 33
    assert relax + moves >= sum(it) * 31 * 31


@pytest.mark.parametrize("shape,levels,omega,nu,mu", [((33, 33), 5, 0.8, (1, 1), 0.6), ((65, 65), 6, 0.8, (2, 1), 0.6),
                                                       ((17, 17, 17), 4, 6 / 7, (1, 1), 5 / 7)])
def test_P11_classic_vcycle(orc, shape, levels, omega, nu, mu):
    rng = np.random.default_rng(8)
    f = rng.standard_normal(shape)
    u, _, norms = orc.vcycle(f, np.zeros(shape), levels, omega, nu[0], nu[1], 25)
    fac = norms[1:] / norms[:-1]
    ok = norms[1:] > 1e-10 * norms[0]
    asym = fac[ok][-1]
    # smoothing-factor estimate mu^(nu1+nu2) from local Fourier analysis, generous band
    est = mu ** sum(nu)
    assert 0.5 * est < asym < 1.35 * est, (asym, est)
    if np.prod(shape) < 5000:
        ud = orc.dense_solve(f)
        u, _, _ = orc.vcycle(f, np.zeros(shape), levels, omega, nu[0], nu[1], 60)
        assert np.abs(u - ud).max() <= 1e-11 * np.abs(ud).max()


def test_P11_vcycle_factor_h_independent(orc):
    facs = []
    for n in (33, 65, 129):
        rng = np.random.default_rng(1)
        f = rng.standard_normal((n, n))
        _, _, norms = orc.vcycle(f, np.zeros((n, n)), int(np.log2(n - 1)), 0.8, 2, 1, 12)
        facs.append(norms[-1] / norms[-2])
    assert max(facs) - min(facs) < 0.03 and 0.15 < facs[-1] < 0.32


def test_cfg1_residual_history_is_reproducible(orc):
    """Per-cycle factors of config 1 (BASELINE.json configs[0]); stored by tests/golden/make_golden.py
    from the oracle alone, here re-derived and compared, plus the structural facts A15 of SURVEY.md."""
    c = I.CONFIGS["cfg1"]
    inp = I.make_inputs(c)
    u, _, n = orc.homg("H", inp["f"], inp["u0"], c.levels, c.omega, orc.schedule(0, c.levels, 4), 10,
                       keep_history=False)
    fac = n[1:] / n[:-1]
    assert fac[0] > 1.0                       # first cycle from u0 = 0 raises the L2 residual (interpolation noise)
    assert np.all(fac[1:] < 0.3) and np.all(fac[1:] > 0.15)
    assert n[-1] / n[0] < 1e-5
    x = np.arange(129) / 128
    uex = np.outer(np.sin(np.pi * x), np.sin(np.pi * x))
    assert np.abs(u - uex).max() < 2e-4       # O(h^2) + noise


def _golden(name):
    import os
    p = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    return np.loadtxt(p, comments="#")


def test_golden_cfg1_norms_match_oracle_and_literal_algorithm(orc):
    gold = _golden("cfg1_norms.txt")
    c = I.CONFIGS["cfg1"]
    inp = I.make_inputs(c)
    sched = orc.schedule(0, c.levels, c.max_iters)
    _, _, nH = orc.homg("H", inp["f"], inp["u0"], c.levels, c.omega, sched, 10, keep_history=False)
    assert np.allclose(nH, gold, rtol=1e-12)
    _, _, nL = orc.homg("L", inp["f"], inp["u0"], c.levels, c.omega, sched, 3, keep_history=False)
    assert np.allclose(nL, gold[:4], rtol=1e-10)
    # ||r_0|| = ||f|| for u0 = 0: independent of the oracle
    inner = (slice(1, -1),) * 2
    assert abs(np.sqrt((inp["f"][inner] ** 2).sum()) - gold[0]) < 1e-12 * gold[0]


def test_golden_paper_L1(orc):
    gold = _golden("paper_L1.txt")
    f, uex = I.paper_polynomial((129, 129))
    for mi, err in gold:
        u, _, _ = orc.homg("H", f, np.zeros((129, 129)), 7, 0.8, orc.schedule(0, 7, int(mi)), 1, keep_history=False)
        mine = np.abs(u - uex).sum() / np.abs(uex).sum()
        assert abs(mine - err) < 0.3 * err, (mi, mine, err)


# ---- mixed-precision outer loop (the restart is a defect-correction loop) ----
@pytest.mark.parametrize("shape,levels,omega,var", [((17, 17), 4, 0.8, False), ((9, 9, 9), 3, 6 / 7, False),
                                                    ((9, 9, 9), 3, 6 / 7, True), ((33, 33), 5, 0.8, False)])
def test_mixed_precision_reaches_the_fp64_fixed_point(orc, shape, levels, omega, var):
    """fp64 residual + fp32 correction cycle converges to the dense-LU solution to fp64 accuracy, where the pure
    fp32 solve stalls at its rounding floor — pins the outer loop (residual in fp64, u += e in fp64)."""
    rng = np.random.default_rng(5)
    f = rng.standard_normal(shape)
    k = np.exp(rng.uniform(-1, 1, shape)) if var else None
    sched = orc.schedule(0, levels, 4)
    ud = orc.dense_solve(f, k=k)
    um, _, nm = orc.homg_mixed(f, np.zeros(shape), levels, omega, sched, 120, k=k, keep_history=False)
    assert np.abs(um - ud).max() <= 1e-11 * np.abs(ud).max()
    assert nm[-1] < 1e-10 * nm[0]
    u32, _, n32 = orc.homg("H", f.astype(np.float32), np.zeros(shape, np.float32), levels, omega, sched, 120,
                           k=None if k is None else k.astype(np.float32), keep_history=False)
    assert np.abs(u32 - ud).max() > 1e-8 * np.abs(ud).max()          # the fp32 floor the mixed loop removes


def test_mixed_precision_contracts_like_fp64(orc):
    """per-cycle residual factors of the mixed loop equal the fp64 cycle's to 3 digits while the residual is above
    the fp32 resolution of one cycle; the first cycle equals the fp32 cycle on the rounded right-hand side."""
    shape, levels, omega = (33, 33, 33), 5, 6 / 7
    rng = np.random.default_rng(6)
    f = rng.standard_normal(shape)
    sched = orc.schedule(0, levels, 4)
    _, _, n64 = orc.homg("H", f, np.zeros(shape), levels, omega, sched, 8, keep_history=False)
    um, hist, nm = orc.homg_mixed(f, np.zeros(shape), levels, omega, sched, 8)
    for c in range(1, 8):
        assert abs(nm[c] / nm[c - 1] - n64[c] / n64[c - 1]) <= 2e-3 * n64[c] / n64[c - 1], c
    # from u = 0 the first residual is f itself: cycle 1 == one fp32 cycle on fl32(f), added in fp64
    u1, _, _ = orc.homg("H", f.astype(np.float32), np.zeros(shape, np.float32), levels, omega, sched, 1, keep_history=False)
    assert np.array_equal(hist[0], u1.astype(np.float64))
