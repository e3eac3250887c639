"""Seeded synthetic inputs for the five BASELINE.json configs (numpy only).

This module serves BOTH the oracle tests and the CUDA path's tests/bench, and for
that reason holds none of the method's arithmetic: no stencil, no relaxation, no
transfer operator.  It only produces right-hand sides, initial guesses and
coefficient fields.

Random numbers come from one counter-based generator: splitmix64 of
(seed, linear node index) -> 53-bit uniform in [0,1); Box-Muller for normals.
Arrays are dense, C order, shape = nodes per axis including the Dirichlet
boundary; coordinates x_a = i_a / (n_a - 1).  Boundary entries of f and u0 are
set to 0 (the solver ignores them anyway).
"""
from dataclasses import dataclass, field

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x):
    """splitmix64 finaliser on a uint64 array (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        z = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def uniform01(seed, n, stream=0, start=0):
    """n uniforms in [0,1): counter = start..start+n-1, keyed by (seed, stream)."""
    with np.errstate(over="ignore"):
        key = _splitmix64(np.array([np.uint64(seed) * np.uint64(0x100000001B3) + np.uint64(stream)], dtype=np.uint64))[0]
        ctr = np.arange(start, start + n, dtype=np.uint64)
        z = _splitmix64(ctr ^ key)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal01(seed, n, chunk=1 << 24):
    """n standard normals by Box-Muller from two uniform streams (chunked to bound memory)."""
    out = np.empty(n, dtype=np.float64)
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        u1 = uniform01(seed, m, stream=1, start=s)
        u2 = uniform01(seed, m, stream=2, start=s)
        out[s:s + m] = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)
    return out


def _zero_boundary(a):
    for ax in range(a.ndim):
        sl = [slice(None)] * a.ndim
        sl[ax] = 0
        a[tuple(sl)] = 0
        sl[ax] = -1
        a[tuple(sl)] = 0
    return a


def coords(shape):
    """list of broadcastable coordinate arrays x_a = i_a/(n_a-1)."""
    out = []
    for ax, n in enumerate(shape):
        sh = [1] * len(shape)
        sh[ax] = n
        out.append((np.arange(n, dtype=np.float64) / (n - 1)).reshape(sh))
    return out


def sine_rhs(shape):
    """f = d*pi^2 * prod sin(pi x_a)  (exact solution of -lap u = f is prod sin(pi x_a))."""
    p = np.ones(shape, dtype=np.float64)
    for x in coords(shape):
        p = p * np.sin(np.pi * x)
    return _zero_boundary(len(shape) * np.pi ** 2 * p)


def uniform_field(shape, seed, lo, hi):
    n = int(np.prod(shape))
    return _zero_boundary((lo + (hi - lo) * uniform01(seed, n)).reshape(shape))


def normal_field(shape, seed):
    return _zero_boundary(normal01(seed, int(np.prod(shape))).reshape(shape))


def fourier_coefficient(shape, seed, nmodes=16):
    """k = exp(g), g = sum of `nmodes` random Fourier modes scaled to max|g| = 1 (R18)."""
    nd = len(shape)
    r = uniform01(seed, nmodes * (nd + 3), stream=7)
    xs = coords(shape)
    g = np.zeros(shape, dtype=np.float64)
    for j in range(nmodes):
        b = r[j * (nd + 3):(j + 1) * (nd + 3)]
        kappa = np.floor(b[:nd] * 9.0).astype(np.int64) - 4          # in {-4..4}
        if not kappa.any():
            kappa[-1] = 1
        amp = np.sqrt(-2.0 * np.log(1.0 - b[nd])) * np.cos(2.0 * np.pi * b[nd + 1])   # N(0,1)
        phase = 2.0 * np.pi * b[nd + 2]
        arg = phase
        for a in range(nd):
            arg = arg + 2.0 * np.pi * float(kappa[a]) * xs[a]
        g += amp * np.cos(arg)
    g /= np.max(np.abs(g))
    return np.exp(g)


def paper_polynomial(shape):
    """PAPER.md Eq.5-6 (2-D): u = -x^2 y^2 (1-x^2)(1-y^2) solves lap u = f_paper.
    Returns (f_spd, u_exact) in the build's convention -lap u = f_spd = -f_paper."""
    y, x = coords(shape)
    u = -(x ** 2) * (y ** 2) * (1 - x ** 2) * (1 - y ** 2)
    fp = -2.0 * (y ** 2 * (1 - 6 * x ** 2) * (1 - y ** 2) + x ** 2 * (1 - 6 * y ** 2) * (1 - x ** 2))
    return _zero_boundary(-fp), _zero_boundary(u)


@dataclass
class Config:
    name: str
    dims: tuple
    levels: int
    dtype: str                 # "f64" | "f32"
    stencil: str               # "poisson5" | "poisson7" | "diffusion7"
    omega: float
    tol: float                 # relative residual to reach (0: fixed cycle count)
    cycles: int                # fixed cycle count when tol == 0, else a cap
    seed: int
    max_iters: int = 4
    schedule: int = 0
    extra: dict = field(default_factory=dict)

    @property
    def np_dtype(self):
        return np.float64 if self.dtype == "f64" else np.float32

    @property
    def n_interior(self):
        return int(np.prod([n - 2 for n in self.dims]))


CONFIGS = {
    "cfg1": Config("cfg1", (129, 129), 7, "f64", "poisson5", 4.0 / 5.0, 0.0, 10, 1),
    "cfg2": Config("cfg2", (129, 129, 129), 7, "f64", "poisson7", 6.0 / 7.0, 1e-8, 40, 2),
    "cfg3": Config("cfg3", (8193, 8193), 13, "f32", "poisson5", 4.0 / 5.0, 1e-5, 40, 3),
    "cfg4": Config("cfg4", (513, 513, 513), 9, "f32", "poisson7", 6.0 / 7.0, 1e-5, 40, 4),
    "cfg5": Config("cfg5", (257, 257, 257), 8, "f64", "diffusion7", 6.0 / 7.0, 1e-8, 60, 5),
}


def scaled(cfg: Config, n: int, levels: int = None) -> Config:
    """The same recipe on an n^d grid (parity tests at sizes the oracle finishes in seconds)."""
    import dataclasses
    import math
    lv = levels if levels is not None else int(round(math.log2(n - 1)))
    return dataclasses.replace(cfg, name=f"{cfg.name}@{n}", dims=(n,) * len(cfg.dims), levels=lv)


def make_inputs(cfg: Config):
    """Returns dict(f=, u0=, k=) as arrays of cfg.np_dtype (k is None for constant coefficient).
    Everything is generated in fp64 and rounded once to the config's dtype."""
    base = cfg.name.split("@")[0]
    shape = tuple(cfg.dims)
    k = None
    u0 = np.zeros(shape, dtype=np.float64)
    if base == "cfg1":
        f = sine_rhs(shape) + uniform_field(shape, cfg.seed, -1e-3, 1e-3)
    elif base == "cfg2":
        f = sine_rhs(shape)
        u0 = uniform_field(shape, cfg.seed, -1.0, 1.0)
    elif base in ("cfg3", "cfg4"):
        f = normal_field(shape, cfg.seed)
    elif base == "cfg5":
        f = _zero_boundary(np.ones(shape, dtype=np.float64))
        k = fourier_coefficient(shape, cfg.seed)
    else:
        raise KeyError(cfg.name)
    dt = cfg.np_dtype
    return {"f": np.ascontiguousarray(f, dtype=dt), "u0": np.ascontiguousarray(u0, dtype=dt),
            "k": None if k is None else np.ascontiguousarray(k, dtype=dt)}
