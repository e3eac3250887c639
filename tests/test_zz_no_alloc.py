"""-m gpu: homg_residual_norm_noalloc (include/homg.h, csrc/homg_noalloc.cu) — the one entry point that allocates
nothing (its per-block partial sums live in a static __device__ array) — against the existing path: a homg_solver
holding the same u and f, homg_residual_norm.  Two (and more) calls in a row share the static scratch: a large grid
first, then a smaller one that leaves the first call's partials behind it, then the large one again.

This file is collected LAST (pytest --collect-only): the suite runs with `pytest -x`, and a failure here must not
hide the parity tests.  It passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from paper_1108_2045_b200 import inputs as I

pytestmark = pytest.mark.gpu

RTOL = {"f64": 1e-10, "f32": 1e-5}          # the tolerances tests/test_gpu_parity.py uses for residual norms


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests")
    return torch


def _case(shape, dtype, seed):
    """u with a zero Dirichlet boundary, f arbitrary inside (seeded, synthetic)."""
    npdt = np.float64 if dtype == "f64" else np.float32
    u = np.ascontiguousarray(I.uniform_field(shape, seed, -1.0, 1.0), dtype=npdt)
    f = np.ascontiguousarray(I.normal_field(shape, seed + 100), dtype=npdt)
    return u, f


def _existing_path(shape, dtype, u, f):
    from paper_1108_2045_b200 import homg
    s = homg.Solver(shape, 1, "poisson5" if len(shape) == 2 else "poisson7", dtype)
    s.set_rhs(f)
    s.set_initial_guess(u)
    norm, _ = s.residual_norm()
    s.destroy()
    return norm


CASES = [((65, 65, 65), "f64", 21), ((33, 33), "f32", 22), ((65, 65, 65), "f64", 23), ((17, 41, 25), "f32", 24),
         ((513, 257), "f64", 25), ((65, 65, 65), "f64", 21)]


def test_no_alloc_residual_norm_matches_the_solver_path_on_calls_in_a_row():
    torch = _torch()
    from paper_1108_2045_b200 import homg
    want = [_existing_path(shape, dtype, *_case(shape, dtype, seed)) for shape, dtype, seed in CASES]
    dev = [tuple(torch.from_numpy(a).cuda() for a in _case(shape, dtype, seed)) for shape, dtype, seed in CASES]
    out = torch.zeros(len(CASES), dtype=torch.float64, device="cuda")
    # calls in a row on one stream, no synchronisation between them: each finds the previous call's partials in the scratch
    for i, (u, f) in enumerate(dev):
        homg.residual_norm_noalloc(u, f, out[i:i + 1])
    got = out.cpu().numpy()
    for (shape, dtype, _), g, w in zip(CASES, got, want):
        assert w > 0 and abs(g - w) <= RTOL[dtype] * w, (shape, dtype, g, w)
    assert got[0] == got[5]                                   # same input, same grid: the same bits (fixed summation order)
    # a second round over the same outputs (the library is warm now): nothing is allocated on the device
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    out2 = out.clone()
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    for i, (u, f) in enumerate(dev):
        homg.residual_norm_noalloc(u, f, out2[i:i + 1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1 <= free0
    assert np.array_equal(out2.cpu().numpy(), got)
    # explicit mesh width
    u, f = dev[1]
    o = torch.zeros(1, dtype=torch.float64, device="cuda")
    homg.residual_norm_noalloc(u, f, o, h=1.0 / 32)
    assert float(o[0]) == got[1]


def test_no_alloc_rejects_sizes_beyond_its_static_scratch():
    torch = _torch()
    from paper_1108_2045_b200 import homg
    import ctypes as C
    L = homg.lib()
    small = torch.zeros(64, dtype=torch.float32, device="cuda")
    o = torch.zeros(1, dtype=torch.float64, device="cuda")
    err = C.create_string_buffer(512)

    def call(dims, dt=homg.HOMG_F32, u=small, f=small, out=o):
        return L.homg_residual_norm_noalloc(len(dims), homg._dims(dims), dt, 0.0, C.c_void_p(u.data_ptr() if u is not None else 0),
                                            C.c_void_p(f.data_ptr() if f is not None else 0),
                                            C.c_void_p(out.data_ptr() if out is not None else 0), None, err, len(err))
    # 513^3 needs 17 * 65 * 513 = 566 865 partials > 131 072: rejected before anything is launched or read
    assert call((513, 513, 513)) == homg.HOMG_EINVAL
    assert b"131072" in err.value and b"566865" in err.value
    assert call((8193, 8193)) == homg.HOMG_EINVAL
    assert call((4, 4, 4, 4)) == homg.HOMG_EINVAL
    assert call((2, 8)) == homg.HOMG_EINVAL
    assert call((8, 8), u=None) == homg.HOMG_EINVAL
    assert call((8, 8), out=None) == homg.HOMG_EINVAL
    assert call((8, 8), dt=2) == homg.HOMG_EINVAL
    assert call((8, 8)) == homg.HOMG_OK                           # 64 scalars: fits the small arrays
    torch.cuda.synchronize()
    assert float(o[0]) == 0.0
    with pytest.raises(homg.HomgError):
        big = torch.zeros((513, 513, 513), dtype=torch.float32, device="cuda")
        homg.residual_norm_noalloc(big, big, o)
