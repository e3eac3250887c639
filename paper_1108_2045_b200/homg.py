"""Thin ctypes binding of libhomg.so (include/homg.h).  Argument marshalling only: every step of
the HOMG cycle runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream.

There is NO CPU fallback: if libhomg.so is missing or cannot be loaded this module raises.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libhomg.so")

HOMG_OK, HOMG_EINVAL, HOMG_ENOMEM, HOMG_ECUDA, HOMG_ESTATE = range(5)
HOMG_F32, HOMG_F64 = 4, 8
HOMG_POISSON5, HOMG_POISSON7, HOMG_DIFFUSION7, HOMG_POISSON5_POW2 = 0, 1, 2, 3
HOMG_SCHED_C, HOMG_SCHED_A, HOMG_SCHED_SAWTOOTH, HOMG_SCHED_EXPLICIT = 0, 1, 2, 3
STENCILS = {"poisson5": HOMG_POISSON5, "poisson7": HOMG_POISSON7, "diffusion7": HOMG_DIFFUSION7,
            "poisson5_pow2": HOMG_POISSON5_POW2}
DTYPES = {"f32": HOMG_F32, "f64": HOMG_F64}

# every symbol include/homg.h declares (tests check that the library exports each one)
SYMBOLS = [
    "homg_default_options", "homg_workspace_bytes", "homg_create", "homg_set_rhs", "homg_set_initial_guess",
    "homg_set_coefficient", "homg_cycle", "homg_solve", "homg_residual_norm", "homg_residual_history", "homg_get_solution",
    "homg_profile_cycles", "homg_tag_name", "homg_compulsory_bytes_per_cycle", "homg_workspace_bytes_mixed", "homg_get_schedule", "homg_launches_per_cycle", "homg_graph_nodes", "homg_bytes_per_cycle", "homg_destroy", "homg_last_error",
    "homg_residual_norm_noalloc",
]


class HomgOptions(C.Structure):
    _fields_ = [
        ("omega", C.c_double), ("h", C.c_double), ("max_iters", C.c_int), ("schedule", C.c_int),
        ("sched_levels", C.POINTER(C.c_int)), ("sched_iters", C.POINTER(C.c_int)), ("sched_len", C.c_int),
        ("coarse_threshold_nodes", C.c_int), ("use_graph", C.c_int), ("history_cap", C.c_int),
        ("tiled_min_nodes", C.c_int), ("march_chunk", C.c_int),
        ("cuda_stream", C.c_void_p), ("cycle", C.c_int), ("v_eta1", C.c_int), ("v_eta2", C.c_int), ("mixed", C.c_int),
    ]


class HomgError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"homg status {status}: {msg}")
        self.status = status


_lib = None


def lib():
    """Loads libhomg.so (never builds, never falls back)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1108_2045_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i, d = C.c_void_p, C.c_int, C.c_double
        i64p = C.POINTER(C.c_int64)
        L.homg_default_options.argtypes = [C.POINTER(HomgOptions)]; L.homg_default_options.restype = None
        L.homg_workspace_bytes.argtypes = [i, i64p, i, i, i]; L.homg_workspace_bytes.restype = C.c_size_t
        L.homg_workspace_bytes_mixed.argtypes = [i, i64p, i, i]; L.homg_workspace_bytes_mixed.restype = C.c_size_t
        L.homg_create.argtypes = [C.POINTER(vp), i, i64p, i, i, i, vp, C.c_size_t, C.POINTER(HomgOptions)]
        L.homg_create.restype = i
        for name in ("homg_set_rhs", "homg_set_initial_guess", "homg_set_coefficient", "homg_get_solution"):
            getattr(L, name).argtypes = [vp, vp, i]; getattr(L, name).restype = i
        L.homg_cycle.argtypes = [vp, i]; L.homg_cycle.restype = i
        L.homg_solve.argtypes = [vp, d, i, C.POINTER(i), C.POINTER(d)]; L.homg_solve.restype = i
        L.homg_residual_norm.argtypes = [vp, C.POINTER(d), C.POINTER(d)]; L.homg_residual_norm.restype = i
        L.homg_residual_history.argtypes = [vp, C.POINTER(d), i, C.POINTER(i)]; L.homg_residual_history.restype = i
        L.homg_get_schedule.argtypes = [vp, C.POINTER(i), C.POINTER(i), i]; L.homg_get_schedule.restype = i
        L.homg_launches_per_cycle.argtypes = [vp]; L.homg_launches_per_cycle.restype = i
        L.homg_graph_nodes.argtypes = [vp, i, C.POINTER(i)]; L.homg_graph_nodes.restype = i
        L.homg_bytes_per_cycle.argtypes = [vp, i]; L.homg_bytes_per_cycle.restype = d
        L.homg_profile_cycles.argtypes = [vp, i, C.POINTER(d), C.POINTER(i), C.POINTER(d), i]; L.homg_profile_cycles.restype = i
        L.homg_tag_name.argtypes = [i]; L.homg_tag_name.restype = C.c_char_p
        L.homg_compulsory_bytes_per_cycle.argtypes = [vp, C.POINTER(d), i]; L.homg_compulsory_bytes_per_cycle.restype = d
        L.homg_destroy.argtypes = [vp]; L.homg_destroy.restype = None
        L.homg_residual_norm_noalloc.argtypes = [i, i64p, i, d, vp, vp, vp, vp, C.c_char_p, C.c_size_t]
        L.homg_residual_norm_noalloc.restype = i
        L.homg_last_error.argtypes = [vp]; L.homg_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _dims(dims):
    return (C.c_int64 * len(dims))(*[int(x) for x in dims])


def workspace_bytes(dims, levels, stencil, dtype):
    return int(lib().homg_workspace_bytes(len(dims), _dims(dims), levels, STENCILS[stencil], DTYPES[dtype]))


def _ptr_and_flag(x):
    """(pointer, on_device) of a torch tensor (CUDA or CPU) or a numpy array; must be C-contiguous."""
    if hasattr(x, "data_ptr"):            # torch.Tensor
        if not x.is_contiguous():
            raise ValueError("array must be contiguous")
        return x.data_ptr(), 1 if x.is_cuda else 0
    if not x.flags["C_CONTIGUOUS"]:
        raise ValueError("array must be C-contiguous")
    return x.ctypes.data, 0


def residual_norm_noalloc(u, f, out, h=0.0, stream=None):
    """homg_residual_norm_noalloc: ||f - A u||_2 of dense CUDA tensors u, f (same shape and dtype, boundary of u = 0)
    into the caller's CUDA float64 tensor `out` (>= 1 element), asynchronously; no allocation by the library (its
    scratch is a static device array: calls that overlap on the GPU race).  Marshalling only."""
    import torch
    if not (u.is_cuda and f.is_cuda and out.is_cuda) or out.dtype != torch.float64 or out.numel() < 1:
        raise ValueError("u, f: CUDA tensors; out: a CUDA float64 tensor")
    if u.shape != f.shape or u.dtype != f.dtype or not (u.is_contiguous() and f.is_contiguous()):
        raise ValueError("u and f must be contiguous tensors of the same shape and dtype")
    dt = {torch.float32: HOMG_F32, torch.float64: HOMG_F64}[u.dtype]
    err = C.create_string_buffer(512)
    with torch.cuda.device(u.device):
        st = stream if stream is not None else torch.cuda.current_stream(u.device)
        rc = lib().homg_residual_norm_noalloc(u.dim(), _dims(tuple(u.shape)), dt, float(h), C.c_void_p(u.data_ptr()),
                                              C.c_void_p(f.data_ptr()), C.c_void_p(out.data_ptr()),
                                              C.c_void_p(st.cuda_stream), err, len(err))
    if rc != HOMG_OK:
        raise HomgError(rc, err.value.decode())


class Solver:
    """homg_create ... homg_destroy.  The workspace is a torch uint8 CUDA tensor owned by this object."""

    def __init__(self, dims, levels, stencil, dtype, omega=0.0, h=0.0, max_iters=0, schedule=HOMG_SCHED_C,
                 sched=None, coarse_threshold_nodes=0, use_graph=-1, history_cap=0, tiled_min_nodes=0,
                 march_chunk=0, device="cuda:0", stream=None, vcycle=None, literal=False, mixed=False):
        import torch
        self._torch = torch
        self.dims = tuple(int(x) for x in dims)
        self.levels = int(levels)
        self.dtype = dtype
        self.handle = C.c_void_p(None)
        L = lib()
        self.device = torch.device(device)
        if self.device.type != "cuda":
            raise ValueError("homg runs on a CUDA device only (no CPU fallback)")
        o = HomgOptions()
        L.homg_default_options(C.byref(o))
        o.omega, o.h, o.max_iters, o.schedule = float(omega), float(h), int(max_iters), int(schedule)
        o.coarse_threshold_nodes, o.use_graph, o.history_cap = int(coarse_threshold_nodes), int(use_graph), int(history_cap)
        o.tiled_min_nodes, o.march_chunk = int(tiled_min_nodes), int(march_chunk)
        if vcycle is not None:                      # classic V(eta1, eta2) instead of the MFMG cycle
            o.cycle, o.v_eta1, o.v_eta2 = 1, int(vcycle[0]), int(vcycle[1])
        if literal:                                 # the paper's whole-grid iteration (Algorithm L)
            o.cycle = 2
        if mixed:                                   # fp64 u, f, residual; the correction cycle in fp32
            o.mixed = 1
        self._keep = None
        if sched is not None:
            lv, it = sched
            a = (C.c_int * len(lv))(*lv); b = (C.c_int * len(it))(*it)
            self._keep = (a, b)
            o.schedule, o.sched_levels, o.sched_iters, o.sched_len = HOMG_SCHED_EXPLICIT, a, b, len(lv)
        with torch.cuda.device(self.device):
            st = stream if stream is not None else torch.cuda.current_stream(self.device)
            o.cuda_stream = C.c_void_p(st.cuda_stream)
            if mixed:
                need = L.homg_workspace_bytes_mixed(len(self.dims), _dims(self.dims), self.levels, STENCILS[stencil])
            else:
                need = L.homg_workspace_bytes(len(self.dims), _dims(self.dims), self.levels, STENCILS[stencil], DTYPES[dtype])
            if need == 0:
                raise HomgError(HOMG_EINVAL, L.homg_last_error(None).decode())
            need += (2 if mixed else 1) * (max(0, int(history_cap) - 4096) * 8 + 256)
            self.workspace = torch.empty(need, dtype=torch.uint8, device=self.device)
            rc = L.homg_create(C.byref(self.handle), len(self.dims), _dims(self.dims), self.levels, STENCILS[stencil],
                               DTYPES[dtype], C.c_void_p(self.workspace.data_ptr()), need, C.byref(o))
        if rc != HOMG_OK:
            self.handle = C.c_void_p(None)
            raise HomgError(rc, L.homg_last_error(None).decode())

    # -- helpers --
    def _ck(self, rc):
        if rc != HOMG_OK:
            raise HomgError(rc, lib().homg_last_error(self.handle).decode())

    def _call_arr(self, fn, x):
        p, dev = _ptr_and_flag(x)
        with self._torch.cuda.device(self.device):
            self._ck(fn(self.handle, C.c_void_p(p), dev))

    # -- the C-ABI calls, same names --
    def set_rhs(self, f):
        self._call_arr(lib().homg_set_rhs, f)

    def set_initial_guess(self, u0):
        """u0 = None: the default guess u = 0 (homg_set_initial_guess with a null pointer)."""
        if u0 is None:
            with self._torch.cuda.device(self.device):
                self._ck(lib().homg_set_initial_guess(self.handle, C.c_void_p(0), 0))
            return
        self._call_arr(lib().homg_set_initial_guess, u0)

    def set_coefficient(self, k):
        self._call_arr(lib().homg_set_coefficient, k)

    def cycle(self, n=1):
        with self._torch.cuda.device(self.device):
            self._ck(lib().homg_cycle(self.handle, int(n)))

    def solve(self, rel_tol, max_cycles):
        """homg_solve: cycles on the device until ||r|| <= rel_tol ||r_0|| or max_cycles; (cycles run, final ||r||/||r_0||)."""
        n = C.c_int(0); r = C.c_double(0)
        with self._torch.cuda.device(self.device):
            self._ck(lib().homg_solve(self.handle, float(rel_tol), int(max_cycles), C.byref(n), C.byref(r)))
        return n.value, r.value

    def residual_norm(self):
        a = C.c_double(0); r = C.c_double(0)
        with self._torch.cuda.device(self.device):
            self._ck(lib().homg_residual_norm(self.handle, C.byref(a), C.byref(r)))
        return a.value, r.value

    def residual_history(self):
        n = C.c_int(0)
        self._ck(lib().homg_residual_history(self.handle, None, 0, C.byref(n)))
        buf = (C.c_double * max(1, n.value))()
        with self._torch.cuda.device(self.device):
            self._ck(lib().homg_residual_history(self.handle, buf, n.value, C.byref(n)))
        return list(buf[:n.value])

    def get_solution(self, out=None):
        if out is None:
            import numpy as np
            out = np.empty(self.dims, dtype=np.float64 if self.dtype == "f64" else np.float32)
        self._call_arr(lib().homg_get_solution, out)
        return out

    def schedule(self):
        n = lib().homg_get_schedule(self.handle, None, None, 0)
        a = (C.c_int * n)(); b = (C.c_int * n)()
        lib().homg_get_schedule(self.handle, a, b, n)
        return list(a), list(b)

    def launches_per_cycle(self):
        return int(lib().homg_launches_per_cycle(self.handle))

    def graph_nodes(self, which=0):
        """node census of the cycle graph (0) or of homg_solve's graph incl. its loop body (1)"""
        c = (C.c_int * 5)()
        self._ck(lib().homg_graph_nodes(self.handle, int(which), c))
        return dict(zip(("kernel", "memset", "memcpy", "conditional", "other"), list(c)))

    def bytes_per_cycle(self, level0_only=False):
        return float(lib().homg_bytes_per_cycle(self.handle, 1 if level0_only else 0))

    def compulsory_bytes_per_cycle(self):
        """{kernel class: bytes the launches of one cycle themselves must move}, and the total."""
        cap = 32
        by = (C.c_double * cap)()
        tot = float(lib().homg_compulsory_bytes_per_cycle(self.handle, by, cap))
        return {lib().homg_tag_name(t).decode(): by[t] for t in range(cap) if lib().homg_tag_name(t) and by[t]}, tot

    def profile_cycles(self, n=1):
        """{kernel class: (total ms, launches, algorithmic bytes)} over n real cycles with per-launch CUDA events."""
        cap = 32
        ms = (C.c_double * cap)(); cnt = (C.c_int * cap)(); by = (C.c_double * cap)()
        with self._torch.cuda.device(self.device):
            self._ck(lib().homg_profile_cycles(self.handle, int(n), ms, cnt, by, cap))
        out = {}
        for t in range(cap):
            name = lib().homg_tag_name(t).decode()
            if name and cnt[t]:
                out[name] = (ms[t], cnt[t], by[t])
        return out

    def destroy(self):
        if self.handle:
            lib().homg_destroy(self.handle)
            self.handle = C.c_void_p(None)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
