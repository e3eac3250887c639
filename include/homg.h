/* homg.h — C ABI of libhomg.so: the high-occupancy multigrid (HOMG) cycle of
 * arxiv 1108.2045 on one B200 (sm_100a).
 *
 * The library solves  A u = f  (Eq.1) with  A = -div(k grad)  on a
 * nested hierarchy of structured grids with Dirichlet u = 0 (Eq.4;
 * the paper writes lap u = f, its f is minus ours — DESIGN.md R1).  One call of
 * homg_cycle runs outer HOMG cycles entirely on the device: residual (L75),
 * nested full-weighting restriction of the residual to every level (L47, L67, L73),
 * the MFMG schedule of whole-level iterations in which the interpolation of the
 * coarse variations and the damped-Jacobi relaxation are one task (L51, L53-71),
 * and the correction u += e (L75).  No host<->device transfer happens inside
 * homg_cycle.
 *
 * Conventions
 *   - dims[a] = nodes per axis INCLUDING the two Dirichlet boundary nodes, dims[0]
 *     slowest (C order).  ndim = 2: (ny, nx); ndim = 3: (nz, ny, nx).
 *   - every dims[a] must equal c_a * 2^(levels-1) + 1 with c_a >= 2 (HOMG_POISSON5_POW2: see there).
 *   - level m = 0 is the finest; level m has (dims[a]-1)/2^m + 1 nodes per axis and
 *     mesh width h_m = 2^m h.
 *   - user arrays (f, u0, k, solution) are DENSE C-order arrays of prod(dims) scalars
 *     of the solver's dtype.  Boundary entries of f and u0 are ignored; the
 *     solution has zeros there.
 *   - "on_device" != 0: the pointer is a CUDA device pointer; 0: a host pointer
 *     (the call then performs the H2D / D2H copy itself, synchronously).
 *   - ownership: the caller owns the workspace and every in/out buffer; the library
 *     owns only its host-side object, CUDA graphs and a few bytes of pinned memory.
 *   - errors: every call returns a homg_status; nothing throws or aborts.  The text
 *     of the last error is available from homg_last_error.
 *   - all device work is issued on the stream given in homg_options.cuda_stream
 *     (NULL = the legacy default stream).
 *   - environment: HOMG_* variables (HOMG_COARSE_NODES, HOMG_COARSE_CLUSTER, HOMG_COARSE_RELAXN,
 *     HOMG_TILED_MIN_NODES, HOMG_MARCH_CHUNK, HOMG_PDL, HOMG_FUSE_FIRST, HOMG_FUSE_FIRST_VAR, HOMG_FUSE_VISIT,
 *     HOMG_VISIT3, HOMG_VISIT_VAR, HOMG_BRICKS, HOMG_DEBUG_SYNC) are read once by homg_create and override the
 *     corresponding homg_options / defaults.  They select between kernels that compute the same cycle (A/B
 *     measurements, the bit-for-bit tests of tests/test_gpu_parity.py); a production caller sets none of them.
 *     HOMG_DEBUG_SYNC synchronises after every launch outside graph capture (to localise a faulting kernel).
 */
#ifndef HOMG_H_
#define HOMG_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define HOMG_API __attribute__((visibility("default")))
#else
#define HOMG_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct homg_solver homg_solver; /* opaque */

typedef enum {
    HOMG_OK = 0,
    HOMG_EINVAL = 1, /* bad argument (dims/levels mismatch, null pointer, bad schedule) */
    HOMG_ENOMEM = 2, /* workspace too small / host allocation failed               */
    HOMG_ECUDA = 3,  /* a CUDA call failed; see homg_last_error                   */
    HOMG_ESTATE = 4  /* call out of order (cycle before set_rhs, ...)             */
} homg_status;

typedef enum { HOMG_F32 = 4, HOMG_F64 = 8 } homg_dtype;

typedef enum {
    HOMG_POISSON5 = 0,  /* 2-D, 5-point  -lap                     (Eq.3) */
    HOMG_POISSON7 = 1,  /* 3-D, 7-point  -lap                     (R10)        */
    HOMG_DIFFUSION7 = 2, /* 3-D, 7-point  -div(k grad), nodal k,
                           harmonic-mean faces, rediscretised per level (R11)  */
    HOMG_POISSON5_POW2 = 3 /* 2-D, 5-point -lap on a grid with a POWER OF TWO number of nodes per side
                           (section 3; R19): dims = (N, N), N = 2^k >= 8,
                           levels <= k.  Four subdomains, coarse points relative to each external corner
                           with the central points just outside every subdomain, same-subdomain
                           interpolation.  Runs the paper's whole-grid iteration (one launch per
                           iteration over the fine grid, as HOMG_CYCLE_LITERAL), whatever `cycle` says.
                           max_iters <= 0 means 32 here (the paper's MaxI of L121): under this reading the
                           contraction per cycle depends on N and MaxI — MaxI = 4: 0.38 at 256^2, 0.84 at
                           1024^2, > 1 (divergence) from 2048^2 on; MaxI = 32: 0.04-0.08 up to 8192^2
                           (R19, measured table in section 11) */
} homg_stencil;

/* MFMG schedule kinds (Fig.1 is missing — DESIGN.md R3).
 * its(m) = min(2^(M-m+1), max_iters), M = levels-1. */
enum {
    HOMG_SCHED_C = 0,        /* M, then for k=M-1..0: k, and if k>0: k+1   (default) */
    HOMG_SCHED_A = 1,        /* M, M-1, then for k=M-2..0: k+2, k+1, k               */
    HOMG_SCHED_SAWTOOTH = 2, /* for k=M..0: M, M-1, .., k                            */
    HOMG_SCHED_EXPLICIT = 3  /* sched_levels / sched_iters, must end on level 0      */
};

typedef struct {
    double omega;     /* weighted-Jacobi damping; <= 0: 4/5 (2-D), 6/7 (3-D)             */
    double h;         /* fine mesh width; <= 0: 1/(dims[0]-1)                            */
    int max_iters;    /* MaxI; <= 0: 4 (HOMG_POISSON5_POW2: 32)           */
    int schedule;     /* HOMG_SCHED_*                                                    */
    const int* sched_levels; /* HOMG_SCHED_EXPLICIT: level of every visit (host ptr)     */
    const int* sched_iters;  /* HOMG_SCHED_EXPLICIT: iterations of every visit, >= 1     */
    int sched_len;
    int coarse_threshold_nodes; /* levels with <= this many nodes run inside the one
                                   persistent coarse-level launch; <= 0: library default */
    int use_graph;    /* 1 (default when < 0): replay one CUDA graph per cycle; 0: plain
                         stream launches (debugging, profiling)                          */
    int history_cap;  /* capacity of the device-side norm history; <= 0: 4096            */
    int tiled_min_nodes; /* levels with >= this many nodes run the TMA-tiled kernels; 0: library
                            default; < 0: never (generic kernels only)                     */
    int march_chunk;  /* planes per CTA along the marching axis of the tiled kernels; <= 0:
                         chosen from the SM count                  */
    void* cuda_stream; /* cudaStream_t; NULL = legacy default stream                     */
    int cycle;        /* HOMG_CYCLE_MFMG (0, default): the paper's high-occupancy cycle;
                         HOMG_CYCLE_V (1): the classic V(v_eta1, v_eta2) cycle of PAPER.md L47 on the
                         same hierarchy, operators and kernels (exact solve on the coarsest level,
                         which must then have exactly one interior node); schedule/max_iters unused;
                         HOMG_CYCLE_LITERAL (2): the paper's own design, same MFMG schedule and same
                         numbers as HOMG_CYCLE_MFMG to rounding, but on ONE fine-grid array with one
                         whole-fine-grid launch per iteration at every level — a
                         measured prior-art row                                                        */
    int v_eta1;       /* pre-smoothing sweeps of HOMG_CYCLE_V; < 0: 2                    */
    int v_eta2;       /* post-smoothing sweeps of HOMG_CYCLE_V; < 0: 1                   */
    int mixed;        /* 1: mixed-precision outer loop (the restart of the cycles is a
                         defect-correction loop).  dtype must be HOMG_F64: u, f, k,
                         the residual r = f - A u and u += e are fp64; r is rounded to fp32 and ONE fp32
                         HOMG cycle on A e = r from e = 0 gives the correction.  The workspace must
                         hold homg_workspace_bytes_mixed() bytes.                                   */
} homg_options;
enum { HOMG_CYCLE_MFMG = 0, HOMG_CYCLE_V = 1, HOMG_CYCLE_LITERAL = 2 };

/* Fills *opt with the defaults (all "use default" markers). */
HOMG_API void homg_default_options(homg_options* opt);

/* Bytes of device workspace a mixed-precision solver (homg_options.mixed = 1) needs: the fp64 level-0
 * arrays plus the fp32 hierarchy (0 on bad arguments). */
HOMG_API size_t homg_workspace_bytes_mixed(int ndim, const int64_t* dims, int levels, homg_stencil stencil);

/* Bytes of device workspace homg_create needs for this hierarchy (0 on bad arguments), for the default
 * history_cap of 4096 entries: a caller that asks for a larger homg_options.history_cap adds
 * (history_cap - 4096) * 8 bytes rounded up to 256 (twice that for a mixed-precision solver).
 * Layout: DESIGN.md "Data layout in HBM" — every level array is contiguous, rows padded
 * to a multiple of 128 bytes, every array 256-byte aligned. */
HOMG_API size_t homg_workspace_bytes(int ndim, const int64_t* dims, int levels, homg_stencil stencil,
                            homg_dtype dtype);

/* Creates a solver over caller-owned device memory [workspace_dev, +workspace_bytes).
 * The workspace is zeroed.  opt may be NULL.  PAPER.md L41-45 (problem), L67 (levels),
 * L69-71 (schedule). */
HOMG_API homg_status homg_create(homg_solver** out, int ndim, const int64_t* dims, int levels,
                        homg_stencil stencil, homg_dtype dtype, void* workspace_dev,
                        size_t workspace_bytes, const homg_options* opt);

/* Right-hand side f (Eq.1).  Resets the norm history. */
HOMG_API homg_status homg_set_rhs(homg_solver* s, const void* f, int on_device);

/* Initial guess u0 (default 0).  u0 == NULL restores the default guess u = 0 on the device (no
 * transfer; on_device is ignored), e.g. before solving again.  Resets the norm history. */
HOMG_API homg_status homg_set_initial_guess(homg_solver* s, const void* u0, int on_device);

/* Nodal coefficient k > 0 (HOMG_DIFFUSION7 only): sampled onto every level by
 * injection (R11).  Must be called before homg_cycle for that stencil. */
HOMG_API homg_status homg_set_coefficient(homg_solver* s, const void* k, int on_device);

/* n outer cycles (residual -> restrict -> MFMG -> u += e), asynchronous on
 * the solver's stream, no host transfers.  Appends n entries to the norm history:
 * entry c = || f - A u ||_2 BEFORE cycle c (sum over interior nodes, accumulated in
 * fp64, no h^d factor — DESIGN.md R12). */
HOMG_API homg_status homg_cycle(homg_solver* s, int n);

/* Cycles until the residual is small: runs outer cycles (as homg_cycle) until
 * || f - A u ||_2 <= rel_tol * || f - A u_0 ||_2  (u_0 = the initial guess: the first history entry) or
 * max_cycles cycles have run — PAPER.md L75: "the residual equation is used to restart the cycles as many
 * times as needed to reach any desired accuracy".  The loop runs ON THE DEVICE: one CUDA graph whose WHILE node
 * repeats the cycle body, the residual-norm kernel at the end of every cycle setting the loop condition; the host
 * is not involved between the launch and the end of the solve (no transfer, no synchronisation inside).  The call
 * then synchronises the stream and reads back the cycle count and two norms (20 bytes).  History: one entry per
 * cycle run (the norm before it), as homg_cycle.  *cycles_done = cycles run by this call, *rel_residual = final
 * || r || / || r_0 || (either may be NULL).  HOMG_CYCLE_MFMG only (plain or mixed precision): HOMG_ESTATE otherwise.
 * HOMG_EINVAL if history_cap < cycles already run + max_cycles + 1. */
HOMG_API homg_status homg_solve(homg_solver* s, double rel_tol, int max_cycles, int* cycles_done, double* rel_residual);

/* PAPER.md L75 ("the residual equation is used to restart the cycles … to reach any desired accuracy"): the accuracy
 * reached.  || f - A u ||_2 of the CURRENT u (one norm-only pass, stream sync, 8-byte D2H) and its
 * ratio to the first history entry (the norm of the initial guess; 1 if no cycle ran).
 * Either output pointer may be NULL. */
HOMG_API homg_status homg_residual_norm(homg_solver* s, double* abs_l2, double* rel_to_initial);

/* The residual norms of the restarts so far (the convergence history of the cycles).
 * Copies min(cap, count) history entries (L2 norms, not squared) to host `out`; syncs. */
HOMG_API homg_status homg_residual_history(homg_solver* s, double* out, int cap, int* count);

/* The solution u of A u = f (Eq. 1) after the cycles run so far, Dirichlet u = 0 on the boundary
 * (L89-93).  Dense C-order copy of u into dst; syncs when dst is a host pointer. */
HOMG_API homg_status homg_get_solution(homg_solver* s, void* dst, int on_device);

/* Introspection for tests and the bench harness: the effective schedule (returns its
 * length; copies at most cap entries), the number of kernel launches one cycle issues,
 * and the algorithmic HBM bytes one cycle moves on level 0 / on all levels
 * (DESIGN.md "Roofline"). */
HOMG_API int homg_get_schedule(const homg_solver* s, int* levels_out, int* iters_out, int cap);
HOMG_API int homg_launches_per_cycle(const homg_solver* s);
/* Node census of the CUDA graph homg_cycle replays (which = 0) or of the graph homg_solve launches, its loop body
 * included (which = 1): counts[0..4] = kernel, memset, memcpy, conditional (WHILE), other nodes.  Evidence for "no
 * host transfers inside a solve": memcpy and other (host, event, ...) are 0.  HOMG_ESTATE before the first
 * homg_cycle / homg_solve. */
HOMG_API homg_status homg_graph_nodes(const homg_solver* s, int which, int* counts);
HOMG_API double homg_bytes_per_cycle(const homg_solver* s, int level0_only);

/* Measurement aid (bench.py): runs n cycles with plain stream launches and a CUDA event after every
 * launch, and accumulates per kernel class the elapsed milliseconds and the launch count into
 * ms_by_tag / launches_by_tag, and the ALGORITHMIC bytes those launches must move (DESIGN.md
 * "Roofline": array passes x nodes x scalar size) into bytes_by_tag (host arrays, cap >= HOMG_TAG_COUNT).  The cycles are real:
 * u advances and n history entries are appended.  Synchronises the stream. */
enum {
    HOMG_TAG_RESIDUAL0 = 0, /* level-0 residual (+norm partials, + first restriction when fused) */
    HOMG_TAG_NORM_FINISH,   /* fixed-order sum of the partials                                    */
    HOMG_TAG_RESTRICT,      /* full weighting g_m = P g_{m-1}                                     */
    HOMG_TAG_RELAX0,        /* level-0 plain Jacobi sweeps                                        */
    HOMG_TAG_RELAX,         /* Jacobi sweeps on levels >= 1                                       */
    HOMG_TAG_DELIVER0,      /* interpolate+correct onto level 0 when not fused into the sweep     */
    HOMG_TAG_DELIVER,       /* interpolate+correct onto levels >= 1                               */
    HOMG_TAG_INJECT,
    HOMG_TAG_D0,            /* carried variation                                                  */
    HOMG_TAG_COARSE,        /* the persistent coarse-level launch                                 */
    HOMG_TAG_OTHER,
    HOMG_TAG_RELAX0_FIRST,  /* level-0 first sweep with interpolate+correct fused (K_relax, first)        */
    HOMG_TAG_RELAX0_LAST,   /* level-0 last sweep of the cycle with u += e fused                          */
    HOMG_TAG_VISIT0,        /* K_visit on level 0: interpolate+correct + all sweeps of the visit + u += e  */
    HOMG_TAG_VISIT,         /* K_visit on levels >= 1: all sweeps of a visit + S3e bookkeeping            */
    HOMG_TAG_COUNT
};
HOMG_API homg_status homg_profile_cycles(homg_solver* s, int n, double* ms_by_tag, int* launches_by_tag,
                                         double* bytes_by_tag, int cap);
HOMG_API const char* homg_tag_name(int tag);
/* COMPULSORY bytes of one cycle per kernel class (bytes_by_tag nullable, cap entries) and their sum
 * (return value): what each launch itself has to move.  Equal to the algorithmic bytes for every
 * single-operation kernel; smaller for K_visit, which performs several Jacobi sweeps (3 arrays each
 * in the per-sweep count of SURVEY.md 8(d)) in one pass.  Valid after the first homg_cycle. */
HOMG_API double homg_compulsory_bytes_per_cycle(const homg_solver* s, double* bytes_by_tag, int cap);

/* The ONE entry point that allocates nothing (csrc/homg_noalloc.cu) — for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it) and hence cannot give a
 * homg_solver its workspace.  The residual-norm step (r = f - A u, ||r||_2 over the interior nodes,
 * accumulated in fp64; A = -lap, 5-point for ndim = 2, 7-point for ndim = 3, mesh width h, h <= 0: 1/(dims[0]-1))
 * of DENSE C-order DEVICE arrays u_dev, f_dev of prod(dims) scalars of `dtype` (dims as everywhere: nodes incl. the
 * boundary, dims[0] slowest).  Boundary entries of u must hold the Dirichlet value 0 (as homg_get_solution returns
 * them); those of f are ignored.  *norm_out_dev (a DEVICE double, caller-owned) receives ||r||_2, asynchronously on
 * cuda_stream (NULL = the legacy default stream); nothing is copied to the host and nothing is synchronised.
 * The per-block partial sums live in a static __device__ array of 131072 doubles (1 MiB, held by every GPU that
 * loads the library until the process exits): a grid with ceil(nx/32) * ceil(ny/8) * nz > 131072 (above 257^3 or
 * 4097^2) is rejected with HOMG_EINVAL.  No cudaMalloc, cudaFree or allocating library routine is called.
 * Every call shares that array: CALLS THAT OVERLAP ON THE GPU (different streams or threads) RACE — serialise
 * them.  Nothing in it needs to start at zero (every block writes its entry; the array keeps the last call's
 * contents).  err (nullable, err_cap bytes) receives the text of an error.  The same value as homg_residual_norm of
 * a solver holding the same u and f, up to the order of the fp64 summation. */
HOMG_API homg_status homg_residual_norm_noalloc(int ndim, const int64_t* dims, homg_dtype dtype, double h,
                                                const void* u_dev, const void* f_dev, double* norm_out_dev,
                                                void* cuda_stream, char* err, size_t err_cap);

HOMG_API void homg_destroy(homg_solver* s);

/* Text of the last error on this solver ("" if none).  s may be NULL: returns the text
 * of the last homg_create failure on this thread. */
HOMG_API const char* homg_last_error(const homg_solver* s);

#ifdef __cplusplus
}
#endif
#endif /* HOMG_H_ */
