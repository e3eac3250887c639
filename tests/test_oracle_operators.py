"""Pins for the oracle's single operators, against closed forms
that the mathematics fixes — never against the oracle's own formulas.

  P2 relaxation   PAPER.md L53-67 (Eq. 2-3): Laplacian eigenvectors, closed-form damping factor
  P3 operator     PAPER.md L41-45 (Eq. 1), L89-93 (Eq. 4): eigenvalues; symmetry, zero row sums (variable k)
  P4 restriction  PAPER.md L47, L73: mode formulas cos^2 / -sin^2
  P5 interpolation PAPER.md L47, L51: exact on multilinear functions; FW = 2^-d S^T; mode formula
"""
import itertools

import numpy as np
import pytest


def mode(shape, kappa):
    """prod_a sin(kappa_a pi x_a) on the nodes of `shape` (zero on the boundary)."""
    v = np.ones(shape)
    for ax, (n, k) in enumerate(zip(shape, kappa)):
        sh = [1] * len(shape)
        sh[ax] = n
        v = v * np.sin(k * np.pi * np.arange(n) / (n - 1)).reshape(sh)
    return v


SHAPES = [(17, 17), (9, 33), (9, 9, 9), (9, 17, 5)]


@pytest.mark.parametrize("shape", SHAPES)
def test_P3_operator_eigenvalues(orc, shape):
    h = 1.0 / (shape[0] - 1)
    for kappa in itertools.product(*[(1, 2, n - 2) for n in shape]):
        v = mode(shape, kappa)
        # axes may have different lengths but share h: eigenvalue uses each axis' own n
        lam = sum(4.0 / h ** 2 * np.sin(k * np.pi / (2 * (n - 1))) ** 2 for k, n in zip(kappa, shape))
        Av = orc.apply_A(v, h=h)
        inner = tuple(slice(1, -1) for _ in shape)
        assert np.allclose(Av[inner], lam * v[inner], rtol=0, atol=1e-10 * lam)
        bmask = np.ones(shape, bool)
        bmask[inner] = False
        assert np.all(Av[bmask] == 0)


@pytest.mark.parametrize("shape,omega", [((17, 17), 0.8), ((9, 33), 0.8), ((9, 9, 9), 6 / 7), ((9, 17, 5), 6 / 7)])
def test_P2_jacobi_damping_factor(orc, shape, omega):
    d = len(shape)
    h = 1.0 / (shape[0] - 1)
    zero = np.zeros(shape)
    for kappa in itertools.product(*[(1, (n - 1) // 2, n - 2) for n in shape]):
        v = mode(shape, kappa)
        fac = 1.0 - (2.0 * omega / d) * sum(np.sin(k * np.pi / (2 * (n - 1))) ** 2 for k, n in zip(kappa, shape))
        out = orc.jacobi(v, zero, omega, h=h)
        assert np.allclose(out, fac * v, rtol=0, atol=1e-13)


def test_P2_smoothing_factor_values(orc):
    # high-frequency maximum of |1 - (2w/d) sum sin^2| : 3/5 (2-D, w=4/5), 5/7 (3-D, w=6/7)
    for d, omega, mu in [(2, 0.8, 3 / 5), (3, 6 / 7, 5 / 7)]:
        n = 65
        shape = (n,) * d
        worst = 0.0
        zero = np.zeros(shape)
        # corners of the high-frequency region: all-highest mode and one-axis-half / others-lowest
        for kappa in [(n - 2,) * d, ((n - 1) // 2,) + (1,) * (d - 1)]:
            v = mode(shape, kappa)
            out = orc.jacobi(v, zero, omega)
            c = tuple(np.unravel_index(np.argmax(np.abs(v)), shape))
            worst = max(worst, abs(out[c] / v[c]))
        assert abs(worst - mu) < 5e-3


def test_P2_jacobi_with_source_fixed_point(orc):
    # v = A^-1 g is a fixed point of the sweep; uses the eigen-relation, not the oracle's A
    shape = (17, 17)
    h = 1 / 16
    v = mode(shape, (2, 3))
    lam = 4 / h ** 2 * (np.sin(2 * np.pi / 32) ** 2 + np.sin(3 * np.pi / 32) ** 2)
    out = orc.jacobi(v, lam * v, 0.8, h=h)
    assert np.allclose(out, v, atol=1e-13)


@pytest.mark.parametrize("shape", [(6, 7), (5, 5, 6)])
def test_P3_variable_coefficient_matrix(orc, shape):
    rng = np.random.default_rng(3)
    k = np.exp(rng.uniform(-1, 1, shape))
    h = 0.37
    A = orc.assemble(shape, h=h, k=k)
    assert np.allclose(A, A.T, rtol=0, atol=1e-12 * np.abs(A).max())
    # positive definite
    assert np.linalg.eigvalsh(0.5 * (A + A.T)).min() > 0
    # rows of nodes with no boundary neighbour sum to zero (constants are in the kernel of -div k grad)
    inner = [n - 2 for n in shape]
    rows = np.arange(A.shape[0]).reshape(inner)
    deep = rows[tuple(slice(1, -1) for _ in shape)].ravel()
    assert deep.size > 0
    assert np.allclose(A[deep].sum(axis=1), 0, atol=1e-12 * np.abs(A).max())
    # an off-diagonal entry is -harmonic mean / h^2 : check one by hand
    p = tuple(2 for _ in shape)
    q = p[:-1] + (3,)
    kf = 2 * k[p] * k[q] / (k[p] + k[q])
    ip = rows[tuple(i - 1 for i in p)]
    iq = rows[tuple(i - 1 for i in q)]
    assert abs(A[ip, iq] + kf / h ** 2) < 1e-12 * kf / h ** 2
    # constant k = c reduces to c * Laplacian
    A1 = orc.assemble(shape, h=h)
    Ac = orc.assemble(shape, h=h, k=np.full(shape, 2.5))
    assert np.allclose(Ac, 2.5 * A1, atol=1e-12 * np.abs(Ac).max())


@pytest.mark.parametrize("shape", [(6, 7), (5, 5, 6), (9, 9), (5, 9, 7)])
def test_P2_variable_coefficient_jacobi_is_v_plus_w_Dinv_residual(orc, shape):
    """PAPER.md L53-57 (Eq. 2, "any elliptic operator") + DESIGN.md R11: the variable-coefficient sweep is
    v + w (g - A v) / diag(A), with A the matrix that P3 pins entry by entry (symmetry, row sums, a hand-computed
    harmonic-mean entry).  The sweep is rebuilt here in numpy from that matrix — its diagonal included — so a
    wrong diagonal in the oracle (e.g. arithmetic instead of harmonic means) fails."""
    rng = np.random.default_rng(11)
    k = np.exp(rng.uniform(-1, 1, shape))
    h, omega = 0.23, 6 / 7 if len(shape) == 3 else 0.8
    A = orc.assemble(shape, h=h, k=k)
    inner = tuple(slice(1, -1) for _ in shape)
    v = np.zeros(shape); g = np.zeros(shape)
    v[inner] = rng.standard_normal([n - 2 for n in shape])
    g[inner] = rng.standard_normal([n - 2 for n in shape]) / h ** 2
    vi, gi = v[inner].ravel(), g[inner].ravel()
    want = vi + omega * (gi - A @ vi) / np.diag(A)
    out = orc.jacobi(v, g, omega, h=h, k=k)
    assert np.allclose(out[inner].ravel(), want, rtol=0, atol=1e-13 * np.abs(want).max())
    bm = np.ones(shape, bool); bm[inner] = False
    assert np.all(out[bm] == 0)
    # the diagonal by hand at one node: sum over the 2d faces of the harmonic means / h^2
    p = tuple(2 for _ in shape)
    D = 0.0
    for a in range(len(shape)):
        for sg in (-1, 1):
            q = tuple(pi + (sg if b == a else 0) for b, pi in enumerate(p))
            D += 2 * k[p] * k[q] / (k[p] + k[q])
    D /= h ** 2
    e = np.zeros(shape); e[p] = 1.0                    # unit impulse, g = 0: out(p) = 1 - w (A e)(p)/D = 1 - w
    assert abs(orc.jacobi(e, np.zeros(shape), omega, h=h, k=k)[p] - (1 - omega)) < 1e-14
    gg = np.zeros(shape); gg[p] = 1.0                  # v = 0, unit source: out(p) = w / D
    assert abs(orc.jacobi(np.zeros(shape), gg, omega, h=h, k=k)[p] - omega / D) < 1e-13 * omega / D
    # the arithmetic-mean mutation must be far outside the tolerance
    Dm = sum((k[p] + k[tuple(pi + (sg if b == a else 0) for b, pi in enumerate(p))]) / 2
             for a in range(len(shape)) for sg in (-1, 1)) / h ** 2
    assert abs(omega / Dm - omega / D) > 1e-4 * omega / D


@pytest.mark.parametrize("shape,omega", [((9, 9), 0.8), ((5, 9, 7), 6 / 7)])
def test_P2_variable_coefficient_jacobi_constant_k(orc, shape, omega):
    """k == c: A = c * (-lap), D = 2d c / h^2, so the sweep equals the constant-coefficient Eq. 3 sweep with
    source g / c, up to rounding; and its modes damp by the P2 closed-form factor."""
    rng = np.random.default_rng(12)
    h, c = 1.0 / (shape[0] - 1), 2.5
    inner = tuple(slice(1, -1) for _ in shape)
    v = np.zeros(shape); g = np.zeros(shape)
    v[inner] = rng.standard_normal([n - 2 for n in shape])
    g[inner] = rng.standard_normal([n - 2 for n in shape]) / h ** 2
    a = orc.jacobi(v, g, omega, h=h, k=np.full(shape, c))
    b = orc.jacobi(v, g / c, omega, h=h)
    assert np.allclose(a, b, rtol=0, atol=1e-13 * np.abs(b).max())
    d = len(shape)
    for kappa in itertools.product(*[(1, n - 2) for n in shape]):
        m = mode(shape, kappa)
        fac = 1.0 - (2.0 * omega / d) * sum(np.sin(kk * np.pi / (2 * (n - 1))) ** 2 for kk, n in zip(kappa, shape))
        out = orc.jacobi(m, np.zeros(shape), omega, h=h, k=np.full(shape, c))
        assert np.allclose(out, fac * m, rtol=0, atol=1e-13)


def test_P3_constant_matrix_entries(orc):
    A = orc.assemble((5, 5), h=0.25)
    assert np.allclose(np.diag(A), 4 / 0.25 ** 2)
    assert A[0, 1] == -16 and A[0, 3] == -16 and A[0, 4] == 0 and A[2, 3] == 0
    A3 = orc.assemble((4, 4, 4), h=0.5)
    assert np.allclose(np.diag(A3), 6 / 0.25)


@pytest.mark.parametrize("shape", [(17, 17), (9, 17), (9, 9, 9), (17, 9, 5)])
def test_P4_restriction_modes(orc, shape):
    cshape = tuple((n - 1) // 2 + 1 for n in shape)
    inner = tuple(slice(1, -1) for _ in shape)
    for kappa in itertools.product(*[(1, 2) for _ in shape]):
        # low mode -> prod cos^2(kappa pi h/2) * coarse mode
        fac = np.prod([np.cos(k * np.pi / (2 * (n - 1))) ** 2 for k, n in zip(kappa, shape)])
        out = orc.restrict(mode(shape, kappa))
        assert np.allclose(out[inner], fac * mode(cshape, kappa)[inner], atol=1e-14)
        # aliasing mode N-kappa on axis 0 -> -sin^2 on that axis
        kal = (shape[0] - 1 - kappa[0],) + tuple(kappa[1:])
        fac2 = -np.sin(kappa[0] * np.pi / (2 * (shape[0] - 1))) ** 2 * np.prod(
            [np.cos(k * np.pi / (2 * (n - 1))) ** 2 for k, n in list(zip(kappa, shape))[1:]])
        out = orc.restrict(mode(shape, kal))
        assert np.allclose(out[inner], fac2 * mode(cshape, kappa)[inner], atol=1e-14)
        bm = np.ones(cshape, bool)
        bm[inner] = False
        assert np.all(out[bm] == 0)


def test_P4_restriction_constants_and_weights(orc):
    out = orc.restrict(np.ones((9, 9)))
    assert np.allclose(out[1:-1, 1:-1], 1.0) and np.all(out[0] == 0) and np.all(out[:, -1] == 0)
    out = orc.restrict(np.ones((9, 9, 9)))
    assert np.allclose(out[1:-1, 1:-1, 1:-1], 1.0)
    # stencil weights from unit impulses: 2-D 4,2,1 over 16; 3-D 8,4,2,1 over 64
    for d in (2, 3):
        shape = (9,) * d
        for off in itertools.product((-1, 0, 1), repeat=d):
            x = np.zeros(shape)
            x[tuple(4 + o for o in off)] = 1.0
            out = orc.restrict(x)
            w = 2.0 ** (-d - sum(abs(o) for o in off))
            assert out[(2,) * d] == w
            assert np.count_nonzero(out) == 2 ** sum(abs(o) for o in off)


@pytest.mark.parametrize("cshape", [(5, 5), (3, 9), (5, 5, 5), (3, 5, 9)])
def test_P5_prolongation_multilinear_exact(orc, cshape):
    fshape = tuple(2 * (n - 1) + 1 for n in cshape)
    d = len(cshape)
    rng = np.random.default_rng(5)
    coef = rng.standard_normal((2,) * d)

    def ml(shape):
        xs = [np.arange(n, dtype=float) / (n - 1) for n in shape]
        g = np.meshgrid(*xs, indexing="ij")
        out = np.zeros(shape)
        for e in itertools.product((0, 1), repeat=d):
            term = coef[e]
            for a in range(d):
                term = term * g[a] ** e[a]
            out = out + term
        return out
    assert np.allclose(orc.prolong(ml(cshape)), ml(fshape), atol=1e-14)
    # identity on coincident nodes, bit for bit
    x = rng.standard_normal(cshape)
    assert np.array_equal(orc.prolong(x)[tuple(slice(None, None, 2) for _ in cshape)], x)


@pytest.mark.parametrize("cshape", [(5, 5), (3, 5), (3, 3, 3), (3, 5, 3)])
def test_P5_restriction_is_scaled_transpose(orc, cshape):
    fshape = tuple(2 * (n - 1) + 1 for n in cshape)
    d = len(cshape)
    nc, nf = int(np.prod(cshape)), int(np.prod(fshape))
    S = np.zeros((nf, nc))
    for j in range(nc):
        e = np.zeros(nc)
        e[j] = 1
        S[:, j] = orc.prolong(e.reshape(cshape)).ravel()
    R = np.zeros((nc, nf))
    for j in range(nf):
        e = np.zeros(nf)
        e[j] = 1
        R[:, j] = orc.restrict(e.reshape(fshape)).ravel()
    cin = np.zeros(cshape, bool)
    cin[tuple(slice(1, -1) for _ in cshape)] = True
    rows = np.flatnonzero(cin.ravel())
    assert np.allclose(R[rows], 2.0 ** (-d) * S.T[rows], atol=1e-15)
    assert np.all(R[np.flatnonzero(~cin.ravel())] == 0)


def test_P5_prolongation_modes(orc):
    # coarse mode kappa -> cos^2 (fine kappa) - sin^2 (fine N-kappa), 1-D factor, tensor in 2-D
    nc, nf = 9, 17
    for kx, ky in [(1, 1), (2, 3), (3, 1)]:
        out = orc.prolong(mode((nc, nc), (kx, ky)))

        def f1(k):
            c = np.cos(k * np.pi / (2 * (nf - 1))) ** 2
            s = np.sin(k * np.pi / (2 * (nf - 1))) ** 2
            x = np.arange(nf) / (nf - 1)
            return c * np.sin(k * np.pi * x) - s * np.sin((nf - 1 - k) * np.pi * x)
        assert np.allclose(out, np.outer(f1(kx), f1(ky)), atol=1e-14)


def test_float32_entry_points_agree_with_float64(orc):
    rng = np.random.default_rng(9)
    for shape in [(17, 17), (9, 9, 9)]:
        v = rng.standard_normal(shape)
        g = rng.standard_normal(shape)
        for fn in (lambda a, b: orc.jacobi(a, b, 0.8), lambda a, b: orc.residual(a, b)[0],
                   lambda a, b: orc.restrict(a), lambda a, b: orc.prolong(a), lambda a, b: orc.apply_A(a)):
            o64 = fn(v, g)
            o32 = fn(v.astype(np.float32), g.astype(np.float32))
            assert o32.dtype == np.float32
            assert np.allclose(o32, o64, rtol=2e-5, atol=2e-5 * np.abs(o64).max())
