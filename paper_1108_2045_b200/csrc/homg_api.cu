// homg_api.cu — the C ABI of libhomg.so (include/homg.h): argument checking, workspace carving,
// graph capture and replay.  No arithmetic of the method happens on the host.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "homg_exec.h"

using namespace homg;

static_assert(int(TAG_COUNT) == int(HOMG_TAG_COUNT), "tag tables out of sync");

namespace {

thread_local std::string g_create_err;

size_t round_up(size_t v, size_t m) { return (v + m - 1) / m * m; }

homg_status set_err(homg_solver* s, homg_status st, const std::string& msg) {
    if (s) s->err = msg; else g_create_err = msg;
    return st;
}

homg_status cuda_fail(homg_solver* s, cudaError_t e, const char* where) {
    return set_err(s, HOMG_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

#define CU(s, call)                                                    \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return cuda_fail((s), e__, #call);     \
    } while (0)

void drop_graph(homg_solver* s) {
    if (s->graph_exec) { cudaGraphExecDestroy(s->graph_exec); s->graph_exec = nullptr; }
    if (s->graph) { cudaGraphDestroy(s->graph); s->graph = nullptr; }
    if (s->solve_exec) { cudaGraphExecDestroy(s->solve_exec); s->solve_exec = nullptr; }
    if (s->solve_graph) { cudaGraphDestroy(s->solve_graph); s->solve_graph = nullptr; }
    s->solve_body = nullptr;
}

cudaError_t census(cudaGraph_t g, int* c) {
    size_t n = 0;
    cudaError_t e = cudaGraphGetNodes(g, nullptr, &n);
    if (e != cudaSuccess) return e;
    std::vector<cudaGraphNode_t> nodes(n + 1);
    if (n && (e = cudaGraphGetNodes(g, nodes.data(), &n)) != cudaSuccess) return e;
    for (size_t i = 0; i < n; ++i) {
        cudaGraphNodeType t;
        if ((e = cudaGraphNodeGetType(nodes[i], &t)) != cudaSuccess) return e;
        if (t == cudaGraphNodeTypeKernel) ++c[0];
        else if (t == cudaGraphNodeTypeMemset) ++c[1];
        else if (t == cudaGraphNodeTypeMemcpy) ++c[2];
        else if (t == cudaGraphNodeTypeConditional) ++c[3];
        else ++c[4];
    }
    return cudaSuccess;
}

struct SolveParamsHost { double tol2; int max_slot; int pad; };   // = SolveParams of homg_kernels.cuh

// homg_solve's graph: [S1 of the initial guess] -> WHILE (norm above tolerance) { S2..S4 of one cycle; S1 of the new u }.
// Both parts are captured from the executor's launch sequence; the norm kernel sets the condition on the device.
homg_status build_solve_graph(homg_solver* s) {
    CU(s, cudaGraphCreate(&s->solve_graph, 0));
    cudaGraphConditionalHandle h;
    cudaError_t e = cudaGraphConditionalHandleCreate(&h, s->solve_graph, 1, cudaGraphCondAssignDefault);
    if (e == cudaSuccess) e = cudaStreamBeginCaptureToGraph(s->cap_stream, s->solve_graph, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) { drop_graph(s); return cuda_fail(s, e, "homg_solve: graph prologue"); }
    e = exec_solve_prologue(s, s->cap_stream, (unsigned long long)h);
    cudaGraph_t got = nullptr;
    cudaError_t e2 = cudaStreamEndCapture(s->cap_stream, &got);
    if (e != cudaSuccess || e2 != cudaSuccess) { drop_graph(s); return cuda_fail(s, e != cudaSuccess ? e : e2, "homg_solve: capture(prologue)"); }
    // the WHILE node depends on the leaves of the prologue
    size_t nn = 0, ne = 0;
    CU(s, cudaGraphGetNodes(s->solve_graph, nullptr, &nn));
    std::vector<cudaGraphNode_t> nodes(nn);
    CU(s, cudaGraphGetNodes(s->solve_graph, nodes.data(), &nn));
    CU(s, cudaGraphGetEdges(s->solve_graph, nullptr, nullptr, &ne));
    std::vector<cudaGraphNode_t> from(ne), to(ne);
    if (ne) CU(s, cudaGraphGetEdges(s->solve_graph, from.data(), to.data(), &ne));
    std::vector<cudaGraphNode_t> leaves;
    for (auto n : nodes) if (std::find(from.begin(), from.end(), n) == from.end()) leaves.push_back(n);
    for (int i = 0; i < 5; ++i) s->solve_census[i] = 0;
    CU(s, census(s->solve_graph, s->solve_census));              // the prologue (before the WHILE node exists)
    cudaGraphNodeParams p = {};
    p.type = cudaGraphNodeTypeConditional;
    p.conditional.handle = h;
    p.conditional.type = cudaGraphCondTypeWhile;
    p.conditional.size = 1;
    cudaGraphNode_t cn;
    e = cudaGraphAddNode(&cn, s->solve_graph, leaves.data(), leaves.size(), &p);
    if (e != cudaSuccess) { drop_graph(s); return cuda_fail(s, e, "homg_solve: conditional node"); }
    cudaGraph_t body = p.conditional.phGraph_out[0];
    s->solve_body = body;
    e = cudaStreamBeginCaptureToGraph(s->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) { drop_graph(s); return cuda_fail(s, e, "homg_solve: graph body"); }
    e = exec_solve_body(s, s->cap_stream, (unsigned long long)h);
    e2 = cudaStreamEndCapture(s->cap_stream, &got);
    if (e != cudaSuccess || e2 != cudaSuccess) { drop_graph(s); return cuda_fail(s, e != cudaSuccess ? e : e2, "homg_solve: capture(body)"); }
    CU(s, census(body, s->solve_census));
    s->solve_census[3] += 1;                                     // the WHILE node itself
    e = cudaGraphInstantiate(&s->solve_exec, s->solve_graph, 0);
    if (e != cudaSuccess) { drop_graph(s); return cuda_fail(s, e, "homg_solve: cudaGraphInstantiate"); }
    return HOMG_OK;
}

homg_status reset_history(homg_solver* s) {
    CU(s, cudaMemsetAsync(s->slot, 0, sizeof(int), s->stream));
    s->cycles_issued = 0;
    return HOMG_OK;
}

// copies a user array (host or device, dense) into a padded level-0 array
homg_status load_dense(homg_solver* s, const void* src, int on_device, void* padded, int zero_boundary) {
    const LevelGeom& g = s->L[0].g;
    size_t bytes = size_t(g.nx) * g.ny * g.nz * size_t(s->dtype);
    const void* dense = src;
    if (!on_device) {
        CU(s, cudaMemcpyAsync(s->staging, src, bytes, cudaMemcpyHostToDevice, s->stream));
        dense = s->staging;
    }
    CU(s, exec_pack(s, s->stream, dense, padded, zero_boundary));
    if (!on_device) CU(s, cudaStreamSynchronize(s->stream));   // the host buffer may be reused on return
    return HOMG_OK;
}

}  // namespace

extern "C" {

void homg_default_options(homg_options* o) {
    if (!o) return;
    std::memset(o, 0, sizeof(*o));
    o->omega = 0; o->h = 0; o->max_iters = 0; o->schedule = HOMG_SCHED_C;
    o->coarse_threshold_nodes = 0; o->use_graph = -1; o->history_cap = 0; o->cuda_stream = nullptr;
    o->cycle = HOMG_CYCLE_MFMG; o->v_eta1 = -1; o->v_eta2 = -1;
}

size_t homg_workspace_bytes(int ndim, const int64_t* dims, int levels, homg_stencil st, homg_dtype dt) {
    Plan P;
    if (!plan_layout(ndim, dims, levels, st, dt, P, &g_create_err)) return 0;
    return P.total_bytes + round_up(size_t(4096) * sizeof(double), 256);   // default history
}

static homg_status create_one(homg_solver** out, int ndim, const int64_t* dims, int levels, homg_stencil st,
                              homg_dtype dt, void* ws, size_t ws_bytes, const homg_options* opt);

size_t homg_workspace_bytes_mixed(int ndim, const int64_t* dims, int levels, homg_stencil st) {
    const size_t a = homg_workspace_bytes(ndim, dims, 1, st, HOMG_F64);
    const size_t b = homg_workspace_bytes(ndim, dims, levels, st, HOMG_F32);
    return (a && b) ? round_up(a, 256) + b : 0;
}

homg_status homg_create(homg_solver** out, int ndim, const int64_t* dims, int levels, homg_stencil st,
                        homg_dtype dt, void* ws, size_t ws_bytes, const homg_options* opt) {
    if (!out) return set_err(nullptr, HOMG_EINVAL, "out is null");
    *out = nullptr;
    if (!opt || !opt->mixed) return create_one(out, ndim, dims, levels, st, dt, ws, ws_bytes, opt);
    // mixed precision: an fp64 one-level outer problem (u, f, r) + the fp32 hierarchy of the correction cycle
    if (dt != HOMG_F64) return set_err(nullptr, HOMG_EINVAL, "mixed precision: dtype must be HOMG_F64 (u, f, k are fp64)");
    if (st == HOMG_POISSON5_POW2) return set_err(nullptr, HOMG_EINVAL, "mixed precision is not available for HOMG_POISSON5_POW2");
    if (opt->cycle != HOMG_CYCLE_MFMG) return set_err(nullptr, HOMG_EINVAL, "mixed precision runs the MFMG cycle only");
    homg_options o = *opt;
    o.mixed = 0;
    const size_t extra = o.history_cap > 4096 ? round_up(size_t(o.history_cap - 4096) * sizeof(double), 256) : 0;
    const size_t a = homg_workspace_bytes(ndim, dims, 1, st, HOMG_F64), b = homg_workspace_bytes(ndim, dims, levels, st, HOMG_F32);
    if (!a || !b) return set_err(nullptr, HOMG_EINVAL, g_create_err);
    const size_t a_al = round_up(a + extra, 256);
    if (!ws) return set_err(nullptr, HOMG_EINVAL, "workspace is null");
    if (ws_bytes < a_al + b + extra) return set_err(nullptr, HOMG_ENOMEM, "workspace too small (see homg_workspace_bytes_mixed)");
    homg_solver* outer = nullptr;
    homg_solver* inner = nullptr;
    homg_status r = create_one(&outer, ndim, dims, 1, st, HOMG_F64, ws, a_al, &o);
    if (r != HOMG_OK) return r;
    r = create_one(&inner, ndim, dims, levels, st, HOMG_F32, static_cast<char*>(ws) + a_al, ws_bytes - a_al, &o);
    if (r != HOMG_OK) { homg_destroy(outer); return r; }
    inner->given_g0 = true;
    outer->inner = inner;
    *out = outer;
    return HOMG_OK;
}

static homg_status create_one(homg_solver** out, int ndim, const int64_t* dims, int levels, homg_stencil st,
                              homg_dtype dt, void* ws, size_t ws_bytes, const homg_options* opt) {
    *out = nullptr;
    Plan P;
    std::string why;
    if (!plan_layout(ndim, dims, levels, st, dt, P, &why)) return set_err(nullptr, HOMG_EINVAL, why);
    if (!ws) return set_err(nullptr, HOMG_EINVAL, "workspace is null");
    homg_options o;
    homg_default_options(&o);
    if (opt) o = *opt;
    int hist_cap = o.history_cap > 0 ? o.history_cap : 4096;
    size_t need = P.total_bytes + round_up(size_t(hist_cap) * sizeof(double), 256);
    if (ws_bytes < need) return set_err(nullptr, HOMG_ENOMEM, "workspace too small (see homg_workspace_bytes)");
    if ((reinterpret_cast<uintptr_t>(ws) & 255) != 0) return set_err(nullptr, HOMG_EINVAL, "workspace must be 256-byte aligned");

    homg_solver* s = new (std::nothrow) homg_solver();
    if (!s) return set_err(nullptr, HOMG_ENOMEM, "host allocation failed");
    s->ndim = ndim; s->levels = levels; s->stencil = st; s->dtype = dt; s->var = P.var;
    s->omega = o.omega > 0 ? o.omega : (ndim == 2 ? 4.0 / 5.0 : 6.0 / 7.0);
    s->h = o.h > 0 ? o.h : 1.0 / double(dims[0] - 1);
    // (power-of-two grids, R19: the contraction of MaxI = 4 degrades with N and is lost from 2048^2 on; the default there is
    // the MaxI = 32 of the paper's own scaling experiment, L121: 0.04-0.08 per cycle up to 8192^2)
    s->max_iters = o.max_iters > 0 ? o.max_iters : (st == HOMG_POISSON5_POW2 ? 32 : 4);
    s->coarse_threshold = o.coarse_threshold_nodes > 0 ? o.coarse_threshold_nodes
                                                       : (o.coarse_threshold_nodes < 0 ? 0 : kCoarseNodesDefault);
    if (const char* ev = std::getenv("HOMG_COARSE_NODES")) s->coarse_threshold = std::atoll(ev);
    if (const char* ev = std::getenv("HOMG_COARSE_CLUSTER")) s->coarse_cluster = std::atoi(ev);
    if (const char* ev = std::getenv("HOMG_COARSE_RELAXN")) s->coarse_relaxn = std::atoi(ev) != 0;
    s->use_graph = o.use_graph != 0;
    s->tiled_min_nodes = o.tiled_min_nodes > 0 ? o.tiled_min_nodes : (o.tiled_min_nodes < 0 ? -1 : kTiledMinNodesDefault);
    if (const char* ev = std::getenv("HOMG_TILED_MIN_NODES")) s->tiled_min_nodes = std::atoll(ev);
    s->march_chunk = o.march_chunk > 0 ? o.march_chunk : 0;
    if (const char* ev = std::getenv("HOMG_MARCH_CHUNK")) s->march_chunk = std::atoi(ev);
    if (const char* ev = std::getenv("HOMG_PDL")) s->pdl = std::atoi(ev) != 0;
    if (const char* ev = std::getenv("HOMG_FUSE_FIRST")) s->fuse_first = std::atoi(ev) != 0;
    if (const char* ev = std::getenv("HOMG_FUSE_FIRST_VAR")) s->fuse_first_var = std::atoi(ev) != 0;
    if (const char* ev = std::getenv("HOMG_FUSE_VISIT")) s->fuse_visit = std::atoi(ev);
    if (const char* ev = std::getenv("HOMG_VISIT3")) s->visit3 = std::atoi(ev);
    if (const char* ev = std::getenv("HOMG_BRICKS")) s->bricks = std::atoi(ev) != 0;
    if (const char* ev = std::getenv("HOMG_VISIT_VAR")) s->visit_var = std::atoi(ev) != 0;
    s->vcycle = o.cycle == HOMG_CYCLE_V;
    s->pow2 = P.pow2;
    s->literal = o.cycle == HOMG_CYCLE_LITERAL || P.pow2;
    if (P.pow2 && o.cycle == HOMG_CYCLE_V) { delete s; return set_err(nullptr, HOMG_EINVAL, "HOMG_POISSON5_POW2 runs the whole-grid HOMG iteration, not the V cycle"); }
    if (P.pow2) s->vcycle = false;
    s->v_eta1 = o.v_eta1 >= 0 ? o.v_eta1 : 2;
    s->v_eta2 = o.v_eta2 >= 0 ? o.v_eta2 : 1;
    s->stream = static_cast<cudaStream_t>(o.cuda_stream);
    s->hist_cap = hist_cap;
    if (build_schedule(o.schedule, levels, s->max_iters, o.sched_levels, o.sched_iters, o.sched_len, s->sched_lv,
                       s->sched_it, &why) < 0) {
        delete s;
        return set_err(nullptr, HOMG_EINVAL, why);
    }
    if (s->vcycle) {
        bool one = true;
        for (int a = 0; a < ndim; ++a) one = one && ((dims[a] - 1) >> (levels - 1)) == 2;
        if (!one || levels < 2) {
            delete s;
            return set_err(nullptr, HOMG_EINVAL, "HOMG_CYCLE_V needs >= 2 levels and a coarsest level of 3 nodes per axis");
        }
    }
    // ---- carve the workspace ----
    s->ws_base = static_cast<char*>(ws); s->ws_bytes = ws_bytes;
    char* p = s->ws_base + 256;             // front guard
    size_t es = size_t(dt);
    auto take = [&](size_t bytes) { void* r = p; p += round_up(bytes, 256); return r; };
    s->L.resize(levels);
    for (int m = 0; m < levels; ++m) {
        Level& L = s->L[m];
        L.g = P.g[m]; L.n_alloc = P.n_alloc[m];
        L.n_nodes = (long long)L.g.nx * L.g.ny * L.g.nz;
        L.h = s->h * double(1LL << m);
        size_t ab = L.n_alloc * es;
        L.nrot = (m == 0) ? 3 : kNumRot;
        if (P.pow2 && m >= 1) {                    // PAPER.md section 3: only the restricted sources live on levels >= 1
            for (int a = 0; a < 4; ++a) s->p2src[a][m] = take(ab);
            L.gsrc = s->p2src[0][m];
            L.nrot = 0;
            continue;
        }
        if (m == 0) { s->u = take(ab); s->f = take(ab); }
        L.gsrc = take(ab);
        for (int b = 0; b < L.nrot; ++b) L.rot[b] = take(ab);
        if (m >= 1) { L.a = take(ab); L.d0 = take(ab); L.tmp = take(ab); }
        if (P.var) { L.k = take(ab); L.fz = take(ab); L.fy = take(ab); L.fx = take(ab); L.wd = take(ab); }
    }
    s->staging = take(P.staging_bytes);
    s->partial = static_cast<double*>(take(P.partial_count * sizeof(double)));
    s->partial_count = P.partial_count;
    s->hist = static_cast<double*>(take(size_t(hist_cap) * sizeof(double)));
    s->slot = static_cast<int*>(take(256));
    s->scalar = reinterpret_cast<double*>(reinterpret_cast<char*>(s->slot) + 128);
    s->solve_params = reinterpret_cast<char*>(s->slot) + 64;
    if (size_t(p - s->ws_base) > ws_bytes) { delete s; return set_err(nullptr, HOMG_ENOMEM, "internal: layout exceeds plan"); }

    cudaError_t e = cudaMemsetAsync(ws, 0, size_t(p - s->ws_base), s->stream);
    if (e == cudaSuccess) e = exec_init(s);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking);
    if (e != cudaSuccess) {
        homg_status r = cuda_fail(nullptr, e, "homg_create");
        delete s;
        return r;
    }
    *out = s;
    return HOMG_OK;
}

homg_status homg_set_rhs(homg_solver* s, const void* f, int on_device) {
    if (!s) return HOMG_EINVAL;
    if (!f) return set_err(s, HOMG_EINVAL, "f is null");
    homg_status r = load_dense(s, f, on_device, s->f, 1);
    if (r != HOMG_OK) return r;
    s->have_rhs = true;
    return reset_history(s);
}

homg_status homg_set_initial_guess(homg_solver* s, const void* u0, int on_device) {
    if (!s) return HOMG_EINVAL;
    if (!u0) {                                         // the default guess u0 = 0: no transfer, one memset
        CU(s, cudaMemsetAsync(s->u, 0, s->L[0].n_alloc * size_t(s->dtype), s->stream));
        return reset_history(s);
    }
    homg_status r = load_dense(s, u0, on_device, s->u, 1);
    if (r != HOMG_OK) return r;
    return reset_history(s);
}

homg_status homg_set_coefficient(homg_solver* s, const void* k, int on_device) {
    if (!s) return HOMG_EINVAL;
    if (!s->var) return set_err(s, HOMG_EINVAL, "this stencil has no coefficient");
    if (!k) return set_err(s, HOMG_EINVAL, "k is null");
    homg_status r = load_dense(s, k, on_device, s->L[0].k, 0);
    if (r != HOMG_OK) return r;
    CU(s, exec_sample_coef(s, s->stream));
    s->have_coef = true;
    if (s->inner) {                                    // the correction cycle uses k rounded to fp32
        CU(s, exec_cvt_coef_to_inner(s, s->stream));
        CU(s, exec_sample_coef(s->inner, s->stream));
        s->inner->have_coef = true;
    }
    return reset_history(s);
}

homg_status homg_cycle(homg_solver* s, int n) {
    if (!s) return HOMG_EINVAL;
    if (n < 0) return set_err(s, HOMG_EINVAL, "n < 0");
    if (!s->have_rhs) return set_err(s, HOMG_ESTATE, "homg_cycle before homg_set_rhs");
    if (s->var && !s->have_coef) return set_err(s, HOMG_ESTATE, "homg_cycle before homg_set_coefficient");
    CU(s, exec_prepare(s));
    if (s->use_graph && !s->graph_exec) {
        // capture one cycle on the private stream (capturing does not execute anything)
        CU(s, cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
        cudaError_t e = exec_cycle(s, s->cap_stream);
        cudaError_t e2 = cudaStreamEndCapture(s->cap_stream, &s->graph);
        if (e != cudaSuccess) { drop_graph(s); return cuda_fail(s, e, "capture(exec_cycle)"); }
        if (e2 != cudaSuccess) { drop_graph(s); return cuda_fail(s, e2, "cudaStreamEndCapture"); }
        e = cudaGraphInstantiate(&s->graph_exec, s->graph, 0);
        if (e != cudaSuccess) { drop_graph(s); return cuda_fail(s, e, "cudaGraphInstantiate"); }
    }
    for (int i = 0; i < n; ++i) {
        if (s->use_graph) CU(s, cudaGraphLaunch(s->graph_exec, s->stream));
        else CU(s, exec_cycle(s, s->stream));
    }
    s->cycles_issued += n;
    return HOMG_OK;
}

homg_status homg_solve(homg_solver* s, double rel_tol, int max_cycles, int* cycles_done, double* rel_residual) {
    if (!s) return HOMG_EINVAL;
    if (!(rel_tol >= 0) || max_cycles < 0) return set_err(s, HOMG_EINVAL, "homg_solve: rel_tol >= 0 and max_cycles >= 0");
    if (!s->have_rhs) return set_err(s, HOMG_ESTATE, "homg_solve before homg_set_rhs");
    if (s->var && !s->have_coef) return set_err(s, HOMG_ESTATE, "homg_solve before homg_set_coefficient");
    if (s->vcycle || s->literal)
        return set_err(s, HOMG_ESTATE, "homg_solve runs the MFMG cycle (HOMG_CYCLE_MFMG, plain or mixed precision); use homg_cycle");
    const long start = s->cycles_issued;
    if (start + max_cycles + 1 > s->hist_cap) return set_err(s, HOMG_EINVAL, "homg_solve: history_cap too small for max_cycles");
    CU(s, exec_prepare(s));
    if (!s->solve_exec) {
        homg_status r = build_solve_graph(s);
        if (r != HOMG_OK) return r;
    }
    SolveParamsHost sp{rel_tol * rel_tol, int(start + max_cycles), 0};
    CU(s, cudaMemcpyAsync(s->solve_params, &sp, sizeof(sp), cudaMemcpyHostToDevice, s->stream));
    CU(s, cudaGraphLaunch(s->solve_exec, s->stream));
    // the solve is over when the stream is: read back how far it went (one int, two doubles)
    int slot = 0;
    CU(s, cudaMemcpyAsync(&slot, s->slot, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
    CU(s, cudaStreamSynchronize(s->stream));
    if (slot < start + 1) return set_err(s, HOMG_ECUDA, "homg_solve: the device loop did not run");
    double n2[2] = {0, 0};
    CU(s, cudaMemcpyAsync(&n2[0], s->hist, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CU(s, cudaMemcpyAsync(&n2[1], s->hist + (slot - 1), sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    // the last entry is the norm of the final u = the norm BEFORE the next cycle: the next cycle records it again
    const int keep = slot - 1;
    CU(s, cudaMemcpyAsync(s->slot, &keep, sizeof(int), cudaMemcpyHostToDevice, s->stream));
    CU(s, cudaStreamSynchronize(s->stream));
    s->cycles_issued = keep;
    if (cycles_done) *cycles_done = int(keep - start);
    if (rel_residual) *rel_residual = n2[0] > 0 ? std::sqrt(n2[1] / n2[0]) : 0.0;
    return HOMG_OK;
}

homg_status homg_residual_norm(homg_solver* s, double* abs_l2, double* rel) {
    if (!s) return HOMG_EINVAL;
    if (!s->have_rhs) return set_err(s, HOMG_ESTATE, "homg_residual_norm before homg_set_rhs");
    CU(s, exec_norm_only(s, s->stream));
    double n2 = 0, first2 = 0;
    CU(s, cudaMemcpyAsync(&n2, s->scalar, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    if (rel && s->cycles_issued > 0)
        CU(s, cudaMemcpyAsync(&first2, s->hist, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CU(s, cudaStreamSynchronize(s->stream));
    double nn = std::sqrt(n2);
    if (abs_l2) *abs_l2 = nn;
    if (rel) *rel = (s->cycles_issued > 0 && first2 > 0) ? nn / std::sqrt(first2) : 1.0;
    return HOMG_OK;
}

homg_status homg_residual_history(homg_solver* s, double* out, int cap, int* count) {
    if (!s) return HOMG_EINVAL;
    long have = s->cycles_issued < s->hist_cap ? s->cycles_issued : s->hist_cap;
    if (count) *count = int(have);
    int n = int(have < cap ? have : cap);
    if (out && n > 0) {
        CU(s, cudaMemcpyAsync(out, s->hist, size_t(n) * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        CU(s, cudaStreamSynchronize(s->stream));
        for (int i = 0; i < n; ++i) out[i] = std::sqrt(out[i]);
    }
    return HOMG_OK;
}

homg_status homg_get_solution(homg_solver* s, void* dst, int on_device) {
    if (!s) return HOMG_EINVAL;
    if (!dst) return set_err(s, HOMG_EINVAL, "dst is null");
    const LevelGeom& g = s->L[0].g;
    size_t bytes = size_t(g.nx) * g.ny * g.nz * size_t(s->dtype);
    if (on_device) {
        CU(s, exec_unpack(s, s->stream, s->u, dst));
    } else {
        CU(s, exec_unpack(s, s->stream, s->u, s->staging));
        CU(s, cudaMemcpyAsync(dst, s->staging, bytes, cudaMemcpyDeviceToHost, s->stream));
        CU(s, cudaStreamSynchronize(s->stream));
    }
    return HOMG_OK;
}

homg_status homg_profile_cycles(homg_solver* s, int n, double* ms_by_tag, int* launches_by_tag,
                                double* bytes_by_tag, int cap) {
    if (!s) return HOMG_EINVAL;
    if (!ms_by_tag || !launches_by_tag || !bytes_by_tag || cap < HOMG_TAG_COUNT) return set_err(s, HOMG_EINVAL, "profile arrays too small");
    if (!s->have_rhs || (s->var && !s->have_coef)) return set_err(s, HOMG_ESTATE, "profile before set_rhs / set_coefficient");
    if (s->inner) return set_err(s, HOMG_ESTATE, "homg_profile_cycles is not available in mixed precision");
    for (int i = 0; i < cap; ++i) { ms_by_tag[i] = 0.0; launches_by_tag[i] = 0; bytes_by_tag[i] = 0.0; }
    CU(s, exec_prepare(s));
    for (int c = 0; c < n; ++c) CU(s, exec_cycle_profiled(s, s->stream, ms_by_tag, launches_by_tag, bytes_by_tag));
    s->cycles_issued += n;
    return HOMG_OK;
}

const char* homg_tag_name(int tag) {
    static const char* names[HOMG_TAG_COUNT] = {"residual_l0", "norm_finish", "restrict", "relax_l0", "relax_coarse",
                                                "deliver_l0", "deliver", "inject", "d0", "coarse_persistent", "other",
                                                "relax_l0_first", "relax_l0_last", "visit_l0", "visit"};
    return (tag >= 0 && tag < HOMG_TAG_COUNT) ? names[tag] : "";
}

int homg_get_schedule(const homg_solver* s, int* lv, int* it, int cap) {
    if (!s) return -1;
    if (s->inner) s = s->inner;
    int n = int(s->sched_lv.size());
    for (int i = 0; i < n && i < cap; ++i) {
        if (lv) lv[i] = s->sched_lv[i];
        if (it) it[i] = s->sched_it[i];
    }
    return n;
}

int homg_launches_per_cycle(const homg_solver* s) { return s ? s->launches_per_cycle : -1; }

homg_status homg_graph_nodes(const homg_solver* s, int which, int* counts) {
    if (!s || !counts) return HOMG_EINVAL;
    for (int i = 0; i < 5; ++i) counts[i] = 0;
    homg_solver* m = const_cast<homg_solver*>(s);
    if (which == 0) {
        if (!s->graph) return set_err(m, HOMG_ESTATE, "homg_graph_nodes before homg_cycle");
        cudaError_t e = census(s->graph, counts);
        return e == cudaSuccess ? HOMG_OK : cuda_fail(m, e, "census(cycle graph)");
    }
    if (!s->solve_graph) return set_err(m, HOMG_ESTATE, "homg_graph_nodes before homg_solve");
    for (int i = 0; i < 5; ++i) counts[i] = s->solve_census[i];   // taken while the graph was built
    return HOMG_OK;
}

double homg_bytes_per_cycle(const homg_solver* s, int level0_only) {
    if (!s) return -1.0;
    return level0_only ? s->bytes_cycle_l0 : s->bytes_cycle_all;
}

double homg_compulsory_bytes_per_cycle(const homg_solver* s, double* bytes_by_tag, int cap) {
    if (!s) return -1.0;
    double tot = 0.0;
    for (int t = 0; t < HOMG_TAG_COUNT; ++t) {
        if (bytes_by_tag && t < cap) bytes_by_tag[t] = s->comp_by_tag[t];
        tot += s->comp_by_tag[t];
    }
    return tot;
}

void homg_destroy(homg_solver* s) {
    if (!s) return;
    if (s->inner) homg_destroy(s->inner);
    drop_graph(s);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    if (s->prog_dev) cudaFree(s->prog_dev);
    delete s;
}

const char* homg_last_error(const homg_solver* s) { return s ? s->err.c_str() : g_create_err.c_str(); }

}  // extern "C"
