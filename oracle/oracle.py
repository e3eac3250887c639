"""ctypes/numpy front end of the C++ oracle (oracle/homg_oracle.cpp).

ORACLE = TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  It holds argument marshalling only;
all arithmetic is in homg_oracle.cpp.  It does not import the CUDA package.
"""
import ctypes as C

import numpy as np

from . import build_oracle

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle.build())
        _lib.orc_assemble.restype = C.c_int64
    return _lib


def _dt(arr):
    if arr.dtype == np.float32:
        return 4
    if arr.dtype == np.float64:
        return 8
    raise TypeError("oracle arrays must be float32 or float64")


def _dims(shape):
    return (C.c_int64 * len(shape))(*shape)


def _p(arr):
    return None if arr is None else arr.ctypes.data_as(C.c_void_p)


def _c(arr, dtype=None):
    if arr is None:
        return None
    return np.ascontiguousarray(arr, dtype=dtype)


def default_h(shape):
    return 1.0 / (shape[0] - 1)


def apply_A(v, h=None, k=None):
    v = _c(v); k = _c(k, v.dtype)
    out = np.empty_like(v)
    rc = lib().orc_apply_A(_dt(v), v.ndim, _dims(v.shape), C.c_double(h or default_h(v.shape)), _p(k), _p(v), _p(out))
    assert rc == 0
    return out


def residual(u, f, h=None, k=None):
    u = _c(u); f = _c(f, u.dtype); k = _c(k, u.dtype)
    r = np.empty_like(u)
    n2 = C.c_double(0)
    rc = lib().orc_residual(_dt(u), u.ndim, _dims(u.shape), C.c_double(h or default_h(u.shape)), _p(k), _p(u), _p(f),
                            _p(r), C.byref(n2))
    assert rc == 0
    return r, float(np.sqrt(n2.value))


def jacobi(v, g, omega, h=None, k=None):
    v = _c(v); g = _c(g, v.dtype); k = _c(k, v.dtype)
    out = np.empty_like(v)
    rc = lib().orc_jacobi(_dt(v), v.ndim, _dims(v.shape), C.c_double(h or default_h(v.shape)), _p(k),
                          C.c_double(omega), _p(v), _p(g), _p(out))
    assert rc == 0
    return out


def restrict(fine):
    fine = _c(fine)
    out = np.empty(tuple((n - 1) // 2 + 1 for n in fine.shape), dtype=fine.dtype)
    rc = lib().orc_restrict(_dt(fine), fine.ndim, _dims(fine.shape), _p(fine), _p(out))
    assert rc == 0
    return out


def prolong(coarse):
    coarse = _c(coarse)
    out = np.empty(tuple(2 * (n - 1) + 1 for n in coarse.shape), dtype=coarse.dtype)
    rc = lib().orc_prolong(_dt(coarse), coarse.ndim, _dims(coarse.shape), _p(coarse), _p(out))
    assert rc == 0
    return out


def schedule(kind, levels, max_iters):
    cap = 4 * levels * levels + 16
    lv = (C.c_int * cap)(); it = (C.c_int * cap)()
    n = lib().orc_schedule(kind, levels, max_iters, lv, it, cap)
    assert n > 0, n
    return list(lv[:n]), list(it[:n])


def _sched_arrays(sched):
    lv, it = sched
    n = len(lv)
    return (C.c_int * n)(*lv), (C.c_int * n)(*it), n


def homg(alg, f, u0, levels, omega, sched, ncycles, h=None, k=None, keep_history=True):
    """ncycles outer HOMG cycles.  alg: 'L' (literal single array) or 'H' (per-level arrays).
    Returns (u, u_hist or None, norms[ncycles+1])."""
    f = _c(f); u = np.array(u0, dtype=f.dtype, order="C", copy=True); k = _c(k, f.dtype)
    hist = np.empty((ncycles,) + f.shape, dtype=f.dtype) if keep_history else None
    norms = np.zeros(ncycles + 1, dtype=np.float64)
    lv, it, n = _sched_arrays(sched)
    rc = lib().orc_homg({"L": 0, "H": 1}[alg], _dt(f), f.ndim, _dims(f.shape), levels,
                        C.c_double(h or default_h(f.shape)), _p(k), C.c_double(omega), lv, it, n, _p(f), _p(u),
                        ncycles, _p(hist), norms.ctypes.data_as(C.POINTER(C.c_double)))
    assert rc == 0, rc
    return u, hist, norms


def homg_mixed(f, u0, levels, omega, sched, ncycles, h=None, k=None, keep_history=True):
    """mixed-precision outer loop: fp64 u, f, residual; one fp32 HOMG cycle (Algorithm H) per
    outer cycle on the residual equation.  Returns (u, u_hist or None, norms[ncycles+1])."""
    f = _c(f, np.float64); u = np.array(u0, dtype=np.float64, order="C", copy=True); k = _c(k, np.float64)
    hist = np.empty((ncycles,) + f.shape, dtype=np.float64) if keep_history else None
    norms = np.zeros(ncycles + 1, dtype=np.float64)
    lv, it, n = _sched_arrays(sched)
    rc = lib().orc_homg_mixed(f.ndim, _dims(f.shape), levels, C.c_double(h or default_h(f.shape)), _p(k),
                              C.c_double(omega), lv, it, n, _p(f), _p(u), ncycles, _p(hist),
                              norms.ctypes.data_as(C.POINTER(C.c_double)))
    assert rc == 0, rc
    return u, hist, norms


def homg_L_partial(f, u0, levels, omega, sched, niters, h=None, k=None):
    """correction array after the first `niters` whole-grid iterations of one literal cycle (fp64)."""
    f = _c(f, np.float64); u = _c(u0, np.float64); k = _c(k, np.float64)
    cur = np.empty_like(f)
    lv, it, n = _sched_arrays(sched)
    rc = lib().orc_homg_L_partial(f.ndim, _dims(f.shape), levels, C.c_double(h or default_h(f.shape)), _p(k),
                                  C.c_double(omega), lv, it, n, _p(f), _p(u), C.c_long(niters), _p(cur))
    assert rc == 0, rc
    return cur


def vcycle(f, u0, levels, omega, eta1, eta2, ncycles, h=None, k=None, keep_history=False):
    f = _c(f); u = np.array(u0, dtype=f.dtype, order="C", copy=True); k = _c(k, f.dtype)
    hist = np.empty((ncycles,) + f.shape, dtype=f.dtype) if keep_history else None
    norms = np.zeros(ncycles + 1, dtype=np.float64)
    rc = lib().orc_vcycle(_dt(f), f.ndim, _dims(f.shape), levels, C.c_double(h or default_h(f.shape)), _p(k),
                          C.c_double(omega), eta1, eta2, _p(f), _p(u), ncycles, _p(hist),
                          norms.ctypes.data_as(C.POINTER(C.c_double)))
    assert rc == 0, rc
    return u, hist, norms


def dense_solve(f, h=None, k=None):
    f = _c(f, np.float64); k = _c(k, np.float64)
    u = np.empty_like(f)
    rc = lib().orc_dense_solve(f.ndim, _dims(f.shape), C.c_double(h or default_h(f.shape)), _p(k), _p(f), _p(u))
    assert rc == 0, rc
    return u


def assemble(shape, h=None, k=None):
    k = _c(k, np.float64)
    N = int(np.prod([n - 2 for n in shape]))
    A = np.empty((N, N), dtype=np.float64)
    rc = lib().orc_assemble(len(shape), _dims(shape), C.c_double(h or default_h(shape)), _p(k), _p(A), C.c_int64(N * N))
    assert rc == N, rc
    return A


def counters(reset=False):
    r = C.c_ulonglong(0); m = C.c_ulonglong(0)
    lib().orc_counters(C.byref(r), C.byref(m), int(reset))
    return r.value, m.value


# ---- Algorithm P: PAPER.md section 3, power-of-two grids (2-D; R19) ----
def homg_p2(f, u0, levels, omega, sched, ncycles, h=None, central=True, keep_history=True):
    f = _c(f); u = np.array(u0, dtype=f.dtype, order="C", copy=True)
    N = f.shape[0]
    assert f.ndim == 2 and f.shape == (N, N)
    hist = np.empty((ncycles, N, N), dtype=f.dtype) if keep_history else None
    norms = np.zeros(ncycles + 1, dtype=np.float64)
    lv, it, n = _sched_arrays(sched)
    rc = lib().orc_homg_p2(_dt(f), C.c_int64(N), levels, C.c_double(h or default_h(f.shape)), C.c_double(omega),
                           int(bool(central)), lv, it, n, _p(f), _p(u), ncycles, _p(hist),
                           norms.ctypes.data_as(C.POINTER(C.c_double)))
    assert rc == 0, rc
    return u, hist, norms


def homg_p2_partial(f, u0, levels, omega, sched, niters, h=None, central=True):
    f = _c(f, np.float64); u = _c(u0, np.float64)
    N = f.shape[0]
    cur = np.empty_like(f)
    lv, it, n = _sched_arrays(sched)
    rc = lib().orc_homg_p2_partial(C.c_int64(N), levels, C.c_double(h or default_h(f.shape)), C.c_double(omega),
                                   int(bool(central)), lv, it, n, _p(f), _p(u), C.c_long(niters), _p(cur))
    assert rc == 0, rc
    return cur


def p2_marked(N, m, central=True):
    mask = np.zeros((N, N), dtype=np.uint8)
    assert lib().orc_p2_marked(C.c_int64(N), m, int(bool(central)), mask.ctypes.data_as(C.c_void_p)) == 0
    return mask.astype(bool)


def p2_iteration(r, cur, prev, levels, m, omega, h=None, central=True):
    r = _c(r, np.float64); cur = _c(cur, np.float64); prev = _c(prev, np.float64)
    N = r.shape[0]
    out = np.empty_like(r)
    rc = lib().orc_p2_iteration(C.c_int64(N), levels, m, C.c_double(h or default_h(r.shape)), C.c_double(omega),
                                int(bool(central)), _p(r), _p(cur), _p(prev), _p(out))
    assert rc == 0, rc
    return out


def p2_restrict(r, levels, m, ay, ax):
    r = _c(r, np.float64)
    N = r.shape[0]
    n = N // (1 << m) + 1
    out = np.empty((n, n), dtype=np.float64)
    assert lib().orc_p2_restrict(C.c_int64(N), levels, m, ay, ax, _p(r), _p(out)) == 0
    return out
