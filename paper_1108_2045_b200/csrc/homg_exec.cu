// homg_exec.cu — the cycle executor: turns the schedule table into the launch sequence of one
// outer HOMG cycle (Algorithm H), issued on a stream (captured once into a CUDA graph
// by homg_api.cu).  Host logic only decides pointers and flags; every arithmetic step is a kernel.
#include "homg_exec.h"

#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include <cstring>
#include <mutex>

#include "homg_coarse.cuh"
#include "homg_first.cuh"
#include "homg_visit.cuh"
#include "homg_visit3.cuh"
#include "homg_moves.cuh"
#include "homg_bricks.cuh"
#include "homg_literal.cuh"
#include "homg_pow2.cuh"

namespace homg {

namespace {

constexpr long long kTinyNodes = 800;   // <= 9^3, 28^2: one CTA works the level (one SM's load bandwidth suffices)

struct Rec {                 // bookkeeping while recording
    homg_solver* s;
    cudaStream_t st;
    cudaError_t err = cudaSuccess;
    int launches = 0;
    double bytes_all = 0, bytes_l0 = 0;
    std::vector<cudaEvent_t>* ev = nullptr;   // profile mode: one event after every launch
    std::vector<int>* ev_tag = nullptr;
    int last_tag = TAG_OTHER;
    double bytes_tag[TAG_COUNT] = {};         // algorithmic bytes per kernel class (per sweep)
    double comp_tag[TAG_COUNT] = {};          // compulsory bytes per kernel class (what the launch must move)
    bool skip_s1 = false;                     // mixed precision: g_0 is given (the rounded fp64 residual), no S1 here
    const void* g_override = nullptr;         // V-cycle, level 0: the sweeps' right-hand side is f, not g_0
    const void* u_override = nullptr;         // V-cycle: the residual is taken of this iterate instead of u
    bool plan = false;                        // planning pass: build the coarse program, launch nothing
    // homg_solve (a CUDA-graph WHILE node loops the cycle on the device): S1 runs at the END of the body on the new
    // u, and its norm kernel sets the loop condition.  Inside a conditional body the first and the last kernel are
    // launched without the programmatic (PDL) attribute (measured: a PDL-attributed last kernel lets the next
    // iteration start early and loses updates).
    bool s1_at_end = false;
    unsigned long long cond = 0;              // cudaGraphConditionalHandle; 0: plain cycle
    bool nopdl_next = false;                  // the next launch carries no PDL attribute
    bool pdl_now() { const bool p = s->pdl && !nopdl_next; nopdl_next = false; return p; }
    std::vector<unsigned char> prog;          // CoarseOp records of the whole cycle, in order
    int prog_nops = 0, run_begin = 0, run_len = 0;
    long long run_maxnodes = 0;
    template <class OP>
    void push(const OP& o, long long nodes) {
        const unsigned char* b = reinterpret_cast<const unsigned char*>(&o);
        prog.insert(prog.end(), b, b + sizeof(OP));
        if (run_len == 0) { run_begin = prog_nops; run_maxnodes = 0; }
        // `act` sits right after `type` in every CoarseOp<T>
        reinterpret_cast<int*>(prog.data() + prog.size() - sizeof(OP))[1] = nodes <= kTinyNodes ? 1 : 0;
        ++prog_nops; ++run_len;
        if (nodes > run_maxnodes) run_maxnodes = nodes;
    }
    void note(cudaError_t e) { if (err == cudaSuccess && e != cudaSuccess) err = e; }
    void acct(int level, double arrays, int tag) { last_tag = tag; acct(level, arrays); }
    // a fused multi-sweep launch: `arrays` = the per-sweep (algorithmic) passes it stands for,
    // `comp` = the passes the fused launch itself has to move
    void acct2(int level, double arrays, double comp, int tag) {
        last_tag = tag;
        acct(level, arrays);
        comp_tag[tag] += (comp - arrays) * double(s->L[level].n_nodes) * double(s->dtype);
    }
    void check(int tag) {
        last_tag = tag;
        if (plan) return;
        cudaError_t e = cudaPeekAtLastError();
        static const bool dbg = std::getenv("HOMG_DEBUG_SYNC") != nullptr;   // localise a faulting launch
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (dbg && e == cudaSuccess && cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs == cudaStreamCaptureStatusNone) {
            e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) std::fprintf(stderr, "homg: launch %d (tag %d) failed: %s\n", launches, tag, cudaGetErrorString(e));
        }
        if (err == cudaSuccess && e != cudaSuccess) err = e;
        ++launches;
        if (ev) {
            cudaEvent_t x;
            cudaEventCreate(&x);
            cudaEventRecord(x, st);
            ev->push_back(x);
            ev_tag->push_back(tag);
        }
    }
    void acct(int level, double arrays) {     // `arrays` passes over one level-`level` array
        double b = arrays * double(s->L[level].n_nodes) * double(s->dtype);
        bytes_all += b;
        bytes_tag[last_tag] += b;
        comp_tag[last_tag] += b;
        if (level == 0) bytes_l0 += b;
    }
};


// every kernel is launched with programmatic stream serialization (PDL): the next kernel of the
// stream / graph may start while this one drains; each kernel executes griddepcontrol.wait before
// its first global access (pdl_start() in homg_kernels.cuh), so data dependences are unchanged.
template <class K, class... Args>
void klaunch(Rec& R, K kern, dim3 grid, dim3 block, size_t smem, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = R.st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = R.pdl_now() ? 1 : 0;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, args...);
    if (R.err == cudaSuccess && e != cudaSuccess) R.err = e;
}

// resident CTAs per SM of a kernel at its launch configuration (asked of the runtime once per kernel): the
// marching-axis chunk counts are chosen so that tiles x chunks fills whole waves of sm_count x this
template <class K>
int resident_ctas(K kern, int threads, size_t smem) {
    // keyed by the kernel's address (one K per signature, one launch configuration per kernel); solvers may be
    // created and cycled from several threads
    static std::mutex mu;
    static std::vector<std::pair<const void*, int>> cache;
    const void* key = reinterpret_cast<const void*>(kern);
    std::lock_guard<std::mutex> lock(mu);
    for (auto& c : cache) if (c.first == key) return c.second;
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, threads, smem) != cudaSuccess || n < 1) n = 1;
    cache.push_back({key, n});
    return n;
}

// level-change kernels: the brick form (homg_bricks.cuh: 2 x 2 fine rows per thread) pays on large fine levels
// (measured: cfg4 1.379 -> 1.366 ms per cycle, cfg5 deliver onto level 0 63 -> 43 us); on small ones its 4 x fewer
// threads cost more latency than the saved loads (cfg2 0.165 -> 0.1725): one pack per thread below 10^6 nodes
inline bool use_bricks(const homg_solver* s, const LevelGeom& gf) {
    return s->bricks && (long long)gf.nx * gf.ny * gf.nz >= 1000000LL;
}
inline dim3 blk() { return dim3(32, 8, 1); }
inline dim3 grd(const LevelGeom& g) { return dim3((g.nx + 31) / 32, (g.ny + 7) / 8, g.nz); }
template <class T>
inline dim3 grdv(const LevelGeom& g) {           // one 16-byte pack of x nodes per thread (homg_moves.cuh)
    const int w = 32 * (16 / int(sizeof(T)));
    return dim3((g.nx + w - 1) / w, (g.ny + 7) / 8, g.nz);
}

template <class T>
Coef<T> make_coef(const homg_solver* s, int m) {
    Coef<T> c;
    double h = s->L[m].h;
    c.ih2 = T(1.0 / (h * h));
    c.w = T(s->omega);
    c.twod = T(2 * s->ndim);
    c.w_over_D = c.w / (c.twod * c.ih2);
    volatile T d = c.twod * c.ih2;          // one rounding, as on the device
    c.D = d;
    volatile T rd = T(1) / d;               // IEEE division: RN(1/D)
    c.rD = rd;
    c.h2 = T(h * h);
    c.wp = T(s->omega / double(2 * s->ndim));
    return c;
}

template <class T>
Faces<T> faces(const Level& L) {
    return Faces<T>{static_cast<const T*>(L.fz), static_cast<const T*>(L.fy), static_cast<const T*>(L.fx)};
}

template <class T>
T* rotp(Level& L, int i) { return i < 0 ? nullptr : static_cast<T*>(L.rot[i]); }


// ---- TMA tensor maps (encoded on the host by the driver's cuTensorMapEncodeTiled) ----------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// map over one level array: dims (nx, ny[, nz]), row pitch px, plane pitch pp; box (bx, by[, 1]).
// Elements outside [0,nx) x [0,ny) x [0,nz) are delivered as 0 (the Dirichlet value / pad).
template <class T, int ND>
bool make_tmap(const homg_solver* s, CUtensorMap* tm, const void* base, const LevelGeom& g, int bx, int by) {
    cuuint64_t gdim[3] = {cuuint64_t(g.nx), cuuint64_t(g.ny), cuuint64_t(g.nz)};
    cuuint64_t gstr[2] = {cuuint64_t(g.px) * sizeof(T), cuuint64_t(g.pp) * sizeof(T)};
    cuuint32_t box[3] = {cuuint32_t(bx), cuuint32_t(by), 1};
    cuuint32_t est[3] = {1, 1, 1};
    CUtensorMapDataType dt = sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    CUresult r = reinterpret_cast<EncodeTiledFn>(s->encode_tiled)(
        tm, dt, ND, const_cast<void*>(base), gdim, gstr, box, est, CU_TENSOR_MAP_INTERLEAVE_NONE,
        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

inline bool tiled(const homg_solver* s, int m) {
    return s->encode_tiled && s->tiled_min_nodes > 0 && s->L[m].n_nodes >= s->tiled_min_nodes;
}

// planes per CTA along the marching axis: as few chunks as fill the machine about once
template <class T, int ND>
int march_chunk(const homg_solver* s, const LevelGeom& g, int* nchunks, int occ = 4) {
    using TL = Tile<T, ND>;
    const int NM = ND == 3 ? g.nz : g.ny;
    const int interior = std::max(NM - 2, 1);
    long long tiles = (long long)((g.nx - 1 + TL::TX - 1) / TL::TX) * (ND == 3 ? (g.ny - 1 + TL::TY - 1) / TL::TY : 1);
    int mc = s->march_chunk;
    if (mc <= 0) {
        long long slots = (long long)s->sm_count * occ;
        long long nch = std::max<long long>(1, slots / std::max<long long>(tiles, 1));
        mc = int((interior + nch - 1) / nch);
        mc = std::max(mc, 8);
    }
    mc = std::min(mc, interior);
    *nchunks = (interior + mc - 1) / mc;
    return mc;
}

// one Jacobi sweep on level t (tiled or generic), with the optional epilogues of k_relax
template <class T, int ND, bool VAR>
void launch_relax(Rec& R, int t, const T* vin, T* vout, T* a, int a_assign, const T* d0, const T* v0, T* u) {
    homg_solver* s = R.s;
    Level& Lt = s->L[t];
    Coef<T> cf = make_coef<T>(s, t);
    if (tiled(s, t)) {
        using TL = Tile<T, ND>;
        CUtensorMap tmv, tmg;
        bool ok = make_tmap<T, ND>(s, &tmv, vin, Lt.g, TL::VW, ND == 3 ? TL::TY + 2 : 1) &&
                  make_tmap<T, ND>(s, &tmg, R.g_override ? R.g_override : Lt.gsrc, Lt.g, TL::SEG, ND == 3 ? TL::TY : 1);
        if (!ok) { if (R.err == cudaSuccess) R.err = cudaErrorInvalidValue; return; }
        int nch = 1;
        int mc = march_chunk<T, ND>(s, Lt.g, &nch, resident_ctas(k_relax_tma<T, ND, VAR>, 256, relax_smem_bytes<T, ND, VAR>()));
        dim3 grid((Lt.g.nx - 1 + TL::TX - 1) / TL::TX, ND == 3 ? (Lt.g.ny - 1 + TL::TY - 1) / TL::TY : nch, ND == 3 ? nch : 1);
        if (u && t == 0) vout = nullptr;              // e_0 is dead after u += e_0: do not write it
        klaunch(R, k_relax_tma<T, ND, VAR>, grid, 256, relax_smem_bytes<T, ND, VAR>(), tmv, tmg, faces<T>(Lt), Lt.g, cf, vout, a, a_assign,
                                                                                      d0, v0, u, mc);
    } else {
        klaunch(R, k_relax<T, ND, VAR>, grd(Lt.g), blk(), 0, Lt.g, cf, vin, (const T*)(R.g_override ? R.g_override : Lt.gsrc), faces<T>(Lt), vout, a,
                                                            a_assign, d0, v0, u);
    }
}


// first sweep of a visit on a tiled level t reached from level t+1 for the first time in the cycle:
// interpolate + correct + relax in one pass (v0 is never written).
template <class T, int ND, bool VAR>
void launch_relax_first(Rec& R, int t, const T* ec, const T* ac, T* vout, T* u) {
    homg_solver* s = R.s;
    Level& Lt = s->L[t];
    Level& Lc = s->L[t + 1];
    using TL = FirstTile<T, ND>;
    CUtensorMap tme, tma_, tmg;
    bool ok = make_tmap<T, ND>(s, &tme, ec, Lc.g, TL::CW, ND == 3 ? TL::CROWS : 1) &&
              make_tmap<T, ND>(s, &tma_, ac, Lc.g, TL::CW, ND == 3 ? TL::CROWS : 1) &&
              make_tmap<T, ND>(s, &tmg, Lt.gsrc, Lt.g, TL::SEG, ND == 3 ? TL::TY : 1);
    if (!ok) { if (R.err == cudaSuccess) R.err = cudaErrorInvalidValue; return; }
    const LevelGeom& g = Lt.g;
    const int NM = ND == 3 ? g.nz : g.ny;
    const int interior = std::max(NM - 2, 1);
    long long tiles = (long long)((g.nx - 1 + TL::TX - 1) / TL::TX) * (ND == 3 ? (g.ny - 1 + TL::TY - 1) / TL::TY : 1);
    int mc = s->march_chunk;
    if (mc <= 0) {
        long long nch = std::max<long long>(1, (long long)s->sm_count * 3 / std::max<long long>(tiles, 1));
        mc = std::max(int((interior + nch - 1) / nch), 8);
    }
    mc = (mc + 1) & ~1;
    int nch = (interior + mc - 1) / mc;
    dim3 grid((g.nx - 1 + TL::TX - 1) / TL::TX, ND == 3 ? (g.ny - 1 + TL::TY - 1) / TL::TY : nch, ND == 3 ? nch : 1);
    klaunch(R, k_relax_first<T, ND, VAR>, grid, TL::NW * 32, first_smem_bytes<T, ND, VAR>(), 
        tme, tma_, tmg, faces<T>(Lt), g, make_coef<T>(s, t), (u && t == 0) ? (T*)nullptr : vout, u, mc);
}


// K_visit: NS sweeps of a visit on a large level in one pass (homg_visit.cuh).
//   interp: stage 0 built from (ec, ac) of level t+1;  otherwise stage 0 = `in` (level t)
template <class T, int ND, int NS, bool INTERP>
void launch_visit(Rec& R, int t, const T* in, const T* ec, const T* ac, T* o0, T* o1, T* o2, T* a, int a_assign,
                  const T* d0, const T* v0, T* u) {
    homg_solver* s = R.s;
    Level& Lt = s->L[t];
    using TL = VisitTile<T, ND, NS>;
    CUtensorMap tm_in, tm_ac, tm_g;
    bool ok = make_tmap<T, ND>(s, &tm_g, R.g_override ? R.g_override : Lt.gsrc, Lt.g, TL::BW, TL::PY);
    if (INTERP) {
        Level& Lc = s->L[t + 1];
        ok = ok && make_tmap<T, ND>(s, &tm_in, ec, Lc.g, TL::CBW, TL::CR) && make_tmap<T, ND>(s, &tm_ac, ac, Lc.g, TL::CBW, TL::CR);
    } else {
        ok = ok && make_tmap<T, ND>(s, &tm_in, in, Lt.g, TL::BW, TL::PY);
        tm_ac = tm_in;
    }
    if (!ok) { if (R.err == cudaSuccess) R.err = cudaErrorInvalidValue; return; }
    const LevelGeom& g = Lt.g;
    const int NM = ND == 3 ? g.nz : g.ny;
    const int interior = std::max(NM - 2, 1);
    const int tx = (g.nx - 1 + TL::OX - 1) / TL::OX, ty = ND == 3 ? (g.ny - 1 + TL::OY - 1) / TL::OY : 1;
    const long long tiles = (long long)tx * ty;
    // chunks of the marching axis: pick the count that minimises waves x (planes per chunk + pipeline fill)
    const bool bookv = !INTERP && (a || o1 || o2);
    const int occ = bookv ? resident_ctas(k_visit<T, ND, NS, false, true>, TL::NT, visit_smem_bytes<T, ND, NS, false>())
                          : resident_ctas(k_visit<T, ND, NS, INTERP, false>, TL::NT, visit_smem_bytes<T, ND, NS, INTERP>());
    const long long slots = (long long)s->sm_count * occ;
    int best = 1;
    double bestc = 1e300;
    for (int nch = 1; nch <= 256 && nch <= interior; ++nch) {
        const int mc = (interior + nch - 1) / nch;
        const long long waves = (tiles * nch + slots - 1) / slots;
        const double c = double(waves) * double(mc + 2 * NS + 6);
        if (c < bestc) { bestc = c; best = nch; }
    }
    int mc = s->march_chunk > 0 ? std::min(s->march_chunk, interior) : (interior + best - 1) / best;
    const int nch = (interior + mc - 1) / mc;
    dim3 grid(tx, ND == 3 ? ty : nch, ND == 3 ? nch : 1);
    if (bookv)
        klaunch(R, k_visit<T, ND, NS, false, true>, grid, TL::NT, visit_smem_bytes<T, ND, NS, false>(), tm_in, tm_ac, tm_g, g,
                make_coef<T>(s, t), o0, o1, o2, a, a_assign, d0, v0, u, mc);
    else
        klaunch(R, k_visit<T, ND, NS, INTERP, false>, grid, TL::NT, visit_smem_bytes<T, ND, NS, INTERP>(), tm_in, tm_ac, tm_g, g,
                make_coef<T>(s, t), o0, o1, o2, a, a_assign, d0, v0, u, mc);
}

// K_visit, 3-D form (homg_visit3.cuh): two rows per thread, g carried in registers
template <class T, int NS, bool INTERP, bool BOOK, bool VAR = false>
void launch_visit3b(Rec& R, int t, const T* in, const T* ec, const T* ac, T* o0, T* o1, T* o2, T* a, int a_assign,
                    const T* d0, const T* v0, T* u) {
    homg_solver* s = R.s;
    Level& Lt = s->L[t];
    using TL = Visit3Tile<T, NS, BOOK, VAR>;
    CUtensorMap tm_in, tm_ac, tm_g, tm_u, tm_fz, tm_fy, tm_fx, tm_wd;
    bool ok = make_tmap<T, 3>(s, &tm_g, R.g_override ? R.g_override : Lt.gsrc, Lt.g, TL::TXN, TL::PY);
    if (INTERP) {
        Level& Lc = s->L[t + 1];
        ok = ok && make_tmap<T, 3>(s, &tm_in, ec, Lc.g, TL::CW, TL::CR) && make_tmap<T, 3>(s, &tm_ac, ac, Lc.g, TL::CW, TL::CR);
    } else {
        ok = ok && make_tmap<T, 3>(s, &tm_in, in, Lt.g, TL::TXN, TL::PY);
        tm_ac = tm_in;
    }
    if (u && !BOOK) ok = ok && make_tmap<T, 3>(s, &tm_u, u, Lt.g, TL::OX, TL::OY);
    else tm_u = tm_g;
    if (VAR) {
        ok = ok && make_tmap<T, 3>(s, &tm_fz, Lt.fz, Lt.g, TL::TXN, TL::PY) && make_tmap<T, 3>(s, &tm_fy, Lt.fy, Lt.g, TL::TXN, TL::PY) &&
             make_tmap<T, 3>(s, &tm_fx, Lt.fx, Lt.g, TL::TXN, TL::PY) && make_tmap<T, 3>(s, &tm_wd, Lt.wd, Lt.g, TL::TXN, TL::PY);
    } else {
        tm_fz = tm_fy = tm_fx = tm_wd = tm_g;
    }
    if (!ok) { if (R.err == cudaSuccess) R.err = cudaErrorInvalidValue; return; }
    const LevelGeom& g = Lt.g;
    const int interior = std::max(g.nz - 2, 1);
    const int tx = (g.nx - 1 + TL::OX - 1) / TL::OX, ty = (g.ny - 1 + TL::OY - 1) / TL::OY;
    const long long tiles = (long long)tx * ty;
    const long long slots = s->sm_count;                           // one CTA per SM
    // z chunks (even length): the count that minimises waves x (planes per chunk + pipeline fill and drain)
    int best = 1;
    double bestc = 1e300;
    for (int nch = 1; nch <= 256 && nch <= std::max(1, interior / 2); ++nch) {
        const int mc = ((interior + nch - 1) / nch + 1) & ~1;
        const int n = (interior + mc - 1) / mc;
        const long long waves = (tiles * n + slots - 1) / slots;
        const double c = double(waves) * double(mc + 2 * NS + 8);
        if (c < bestc) { bestc = c; best = nch; }
    }
    int mc = s->march_chunk > 0 ? std::min(s->march_chunk, interior) : (interior + best - 1) / best;
    mc = (mc + 1) & ~1;
    const int nch = (interior + mc - 1) / mc;
    dim3 grid(tx, ty, nch);
    klaunch(R, k_visit3<T, NS, INTERP, BOOK, VAR>, grid, TL::NT, visit3_smem_bytes<T, NS, INTERP, BOOK, VAR>(), tm_in, tm_ac, tm_g, tm_u,
            tm_fz, tm_fy, tm_fx, tm_wd, g, make_coef<T>(s, t), o0, o1, o2, a, a_assign, d0, v0, u, mc);
}
template <class T, int NS, bool INTERP>
void launch_visit3(Rec& R, int t, const T* in, const T* ec, const T* ac, T* o0, T* o1, T* o2, T* a, int a_assign,
                   const T* d0, const T* v0, T* u) {
    if (!INTERP && (a || o1 || o2)) launch_visit3b<T, NS, false, true>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
    else launch_visit3b<T, NS, INTERP, false>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
}

template <class T, int ND, bool INTERP, bool VAR = false>
void launch_visit_ns(Rec& R, int ns, int t, const T* in, const T* ec, const T* ac, T* o0, T* o1, T* o2, T* a,
                     int a_assign, const T* d0, const T* v0, T* u) {
    if (VAR) {                                    // variable coefficient: 3-D, level-0 form, two sweeps per pass
        if (ND == 3 && ns == 2 && !(a || o1 || o2)) launch_visit3b<T, 2, INTERP, false, ND == 3 && VAR>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
        else if (R.err == cudaSuccess) R.err = cudaErrorInvalidValue;
        return;
    }
    // (visit3 == 1 keeps the S3e-bookkeeping form of levels >= 1 on homg_visit.cuh)
    if (ND == 3 && R.s->visit3 && (R.s->visit3 >= 2 || INTERP || !(a || o1 || o2))) {
        if (ns == 2) launch_visit3<T, 2, INTERP>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
        else if (ns == 3) launch_visit3<T, 3, INTERP>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
        else launch_visit3<T, 4, INTERP>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
        return;
    }
    if (ns == 2) launch_visit<T, ND, 2, INTERP>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
    else if (ns == 3) launch_visit<T, ND, 3, INTERP>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
    else launch_visit<T, ND, 4, INTERP>(R, t, in, ec, ac, o0, o1, o2, a, a_assign, d0, v0, u);
}

// launches the pending run of coarse-level operations as ONE cluster (K_coarse)
template <class T, int ND, bool VAR>
void flush_run(Rec& R) {
    if (R.run_len == 0) return;
    homg_solver* s = R.s;
    if (!R.plan) {
        int ncta = R.run_maxnodes <= kTinyNodes ? 1 : 8;
        if (s->coarse_cluster > 0) ncta = s->coarse_cluster;
        for (int b = 0; b < R.run_len; b += kMaxRunOps) {       // long runs: kMaxRunOps records per launch
            const int n = std::min(kMaxRunOps, R.run_len - b);
            const CoarseOp<T>* dev = static_cast<const CoarseOp<T>*>(s->prog_dev) + R.run_begin + b;
            size_t smem = 0;                                     // OP_RELAXN: 3 compact copies of its level
            {
                const CoarseOp<T>* hops = reinterpret_cast<const CoarseOp<T>*>(R.prog.data()) + R.run_begin + b;
                for (int i = 0; i < n; ++i)
                    if (hops[i].type == OP_RELAXN)
                        smem = std::max(smem, 3 * size_t(hops[i].go.nx) * hops[i].go.ny * hops[i].go.nz * sizeof(T));
            }
            cudaLaunchConfig_t cfg = {};
            cfg.dynamicSmemBytes = smem;
            cfg.gridDim = dim3(ncta, 1, 1);
            cfg.blockDim = dim3(1024, 1, 1);
            cfg.stream = R.st;
            cudaLaunchAttribute at[2];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = ncta; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            at[1].val.programmaticStreamSerializationAllowed = R.pdl_now() ? 1 : 0;
            cfg.attrs = at; cfg.numAttrs = 2;
            cudaError_t e = ncta > 1 ? cudaLaunchKernelEx(&cfg, k_coarse_run<T, ND, VAR, true>, dev, n)
                                     : cudaLaunchKernelEx(&cfg, k_coarse_run<T, ND, VAR, false>, dev, n);
            if (R.err == cudaSuccess && e != cudaSuccess) R.err = e;
            R.check(TAG_COARSE);
        }
    }
    R.run_len = 0;
}

// S1 (+S5, + first step of S2 when `restrict1`): r = f - A u, ||r||^2 -> history / scalar, g_1 = P r.
// Returns true when g_1 was written by the fused kernel.
template <class T, int ND, bool VAR>
bool rec_norm(Rec& R, bool write_r, bool to_history, bool restrict1 = false) {
    homg_solver* s = R.s;
    Level& L0 = s->L[0];
    int n = 0;
    bool fused_restrict = false;
    if (tiled(s, 0)) {
        using TL = ResTile<T, ND>;
        CUtensorMap tmu, tmf;
        bool ok = make_tmap<T, ND>(s, &tmu, R.u_override ? R.u_override : s->u, L0.g, TL::UW, ND == 3 ? TL::TY + 3 : 1) &&
                  make_tmap<T, ND>(s, &tmf, s->f, L0.g, TL::SEG, ND == 3 ? TL::TY + 1 : 1);
        if (!ok) { if (R.err == cudaSuccess) R.err = cudaErrorInvalidValue; return false; }
        fused_restrict = restrict1 && write_r && s->levels >= 2;
        const LevelGeom& g = L0.g;
        const int NM = ND == 3 ? g.nz : g.ny;
        const int interior = std::max(NM - 2, 1);
        long long tiles = (long long)((g.nx - 1 + TL::TX - 1) / TL::TX) * (ND == 3 ? (g.ny - 1 + TL::TY - 1) / TL::TY : 1);
        int mc = s->march_chunk;
        if (mc <= 0) {
            // chunk count: fill whole waves of (148 x resident CTAs) as evenly as possible — an SM with fewer CTAs than
            // its residency cannot draw its share of the bandwidth — at little halo overhead (2 planes per chunk)
            const int occ = resident_ctas(k_res_tma<T, ND, VAR>, TL::NW * 32, res_smem_bytes<T, ND, VAR>());
            const long long slots = (long long)s->sm_count * occ;
            // (one wave that fills >= 80 % of the slots is kept: measured best on cfg3 / cfg5; cfg4's 256 tiles fill 58 %)
            double best = -1.0, best1 = -1.0;
            int bestn = 1, bestn1 = 1;
            for (int nch = 1; nch <= std::max(1, interior / 8); ++nch) {
                const int m = (interior + nch - 1) / nch;
                const long long ctas = tiles * nch, waves = (ctas + slots - 1) / slots;
                const double score = double(ctas) / double(waves * slots) * double(m) / double(m + 2);
                if (score > best + 1e-9) { best = score; bestn = nch; }
                if (waves == 1 && score > best1 + 1e-9) { best1 = score; bestn1 = nch; }
                if (waves > 8) break;
            }
            if (best1 >= 0.8) bestn = bestn1;
            mc = (interior + bestn - 1) / bestn;
        }
        mc = (mc + 1) & ~1;                                        // even: chunks start on odd planes
        int nch = (interior + mc - 1) / mc;
        dim3 grid((g.nx - 1 + TL::TX - 1) / TL::TX, ND == 3 ? (g.ny - 1 + TL::TY - 1) / TL::TY : nch, ND == 3 ? nch : 1);
        n = int(grid.x * grid.y * grid.z);
        if (!R.plan) klaunch(R, k_res_tma<T, ND, VAR>, grid, TL::NW * 32, res_smem_bytes<T, ND, VAR>(), 
            tmu, tmf, faces<T>(L0), g, fused_restrict ? s->L[1].g : g, make_coef<T>(s, 0), write_r ? (T*)L0.gsrc : nullptr,
            fused_restrict ? (T*)s->L[1].gsrc : nullptr, s->partial, mc);
        R.check(TAG_RESIDUAL0);
        R.acct(0, (write_r ? 3.0 : 2.0) + (VAR ? 3.0 : 0.0));
        if (fused_restrict) R.acct(1, 1.0);
    } else {
        dim3 g = grd(L0.g);
        if (!R.plan) klaunch(R, k_residual<T, ND, VAR>, g, blk(), 0, L0.g, make_coef<T>(s, 0), (const T*)(R.u_override ? R.u_override : s->u), (const T*)s->f,
                                                       faces<T>(L0), write_r ? (T*)L0.gsrc : nullptr, s->partial);
        R.check(TAG_RESIDUAL0);
        R.acct(0, (write_r ? 3.0 : 2.0) + (VAR ? 3.0 : 0.0));
        n = int(g.x * g.y * g.z);
    }
    if (!R.plan) {
        if (R.cond) {                                            // homg_solve: the norm decides whether the loop goes on
            R.nopdl_next = true;
            klaunch(R, k_norm_finish_solve, 1, 256, 0, s->partial, n, s->hist, s->slot, s->hist_cap, (const SolveParams*)s->solve_params,
                    R.cond);
        } else {
            klaunch(R, k_norm_finish, 1, 256, 0, s->partial, n, to_history ? s->hist : nullptr, s->slot, s->hist_cap,
                    to_history ? 1 : 0, to_history ? nullptr : s->scalar);
        }
    }
    R.check(TAG_NORM_FINISH);
    return fused_restrict;
}

template <class T, int ND, bool VAR>
void rec_cycle(Rec& R) {
    homg_solver* s = R.s;
    const int M = s->levels - 1;
    std::vector<Level>& L = s->L;
    for (auto& l : L) { l.e = 0; l.touched = false; l.vk = l.vkm1 = l.vkm2 = -1; l.eta_last = 0; }
    std::vector<char> a_zero(s->levels, 1);      // a_m == 0 (nothing pending)
    std::vector<char> dp_is_d0(s->levels, 0);    // eta == 1 visit: its dp is its own d0
    auto small = [&](int m) { return s->coarse_threshold > 0 && L[m].n_nodes <= s->coarse_threshold; };
    auto newop = [&](int type, int mo) {
        CoarseOp<T> o;
        std::memset(&o, 0, sizeof(o));
        o.type = type; o.go = L[mo].g; o.gi = L[mo].g; o.gv = L[mo].g;
        return o;
    };
    auto flush = [&]() { flush_run<T, ND, VAR>(R); };

    // S1: r = f - A u, ||r||^2 -> history
    // (homg_solve: S1 of this cycle ran at the end of the previous loop body, or in the prologue)
    if (R.s1_at_end) R.nopdl_next = true;
    const bool have_g1 = R.skip_s1 ? false : R.s1_at_end ? (tiled(s, 0) && s->levels >= 2) : rec_norm<T, ND, VAR>(R, true, true, true);
    // S2: nested restriction g_m = P g_{m-1}
    for (int m = have_g1 ? 2 : 1; m <= M; ++m) {
        if (small(m)) {
            CoarseOp<T> o = newop(OP_RESTRICT, m);
            o.gi = L[m - 1].g; o.p[0] = (const T*)L[m - 1].gsrc; o.q[0] = (T*)L[m].gsrc;
            R.push(o, L[m].n_nodes);
        } else {
            flush();
            if (!R.plan) klaunch(R, k_restrict<T, ND>, grd(L[m].g), blk(), 0, L[m].g, L[m - 1].g, (const T*)L[m - 1].gsrc, (T*)L[m].gsrc);
            R.check(TAG_RESTRICT);
        }
        R.acct(m - 1, 1.0, small(m) ? TAG_COARSE : TAG_RESTRICT); R.acct(m, 1.0, small(m) ? TAG_COARSE : TAG_RESTRICT);
    }
    // S3: MFMG visits
    int cur = -1;
    const int nv = int(s->sched_lv.size());
    for (int vi = 0; vi < nv; ++vi) {
        const int t = s->sched_lv[vi], eta = s->sched_it[vi];
        Level& Lt = L[t];
        bool have_d0 = false;
        bool fuse_first = false;
        const T* fuse_ec = nullptr;
        // K_visit runs this visit (decided here because a level-0 visit in MID-cycle must leave v^{eta-1} behind for
        // the carried variation of the next visit: K_visit stores it only in its bookkeeping form, which takes its
        // v^0 from memory — such a visit is not fused with its arrival)
        // (variable coefficient, 8(f)4b: K_visit's level-0 form only, two sweeps per pass, when visit_var is on; not in the
        // fp32 inner cycle of the mixed-precision loop, whose parity with the mixed oracle rests on bit-exact sweeps)
        const int kv_maxns = VAR ? 2 : std::min(s->fuse_visit, 4);
        const bool mid_l0 = t == 0 && vi != nv - 1;
        const bool use_kvisit = (VAR ? (ND == 3 && s->visit_var && !s->given_g0 && s->visit3 && t == 0 && !mid_l0) : true) && std::min(s->fuse_visit, 4) >= 2 &&
                                tiled(s, t) && !(s->coarse_threshold > 0 && Lt.n_nodes <= s->coarse_threshold) &&
                                eta >= 2 && (t == 0 || eta <= kv_maxns);
        if (cur < 0) {
            if (small(t)) {
                CoarseOp<T> o = newop(OP_ZERO, t);
                o.count = (long long)Lt.n_alloc; o.q[0] = (T*)Lt.rot[Lt.e];
                R.push(o, L[t].n_nodes);
            } else {
                flush();
                if (!R.plan) R.note(cudaMemsetAsync(Lt.rot[Lt.e], 0, Lt.n_alloc * sizeof(T), R.st));
                R.check(TAG_OTHER);
            }
            Lt.touched = true;
        } else {
            // a deliver onto a large level whose hop also carries a step of the S3c prolongation (t >= 1) is
            // held back and launched together with it (k_arrive_v): one launch per hop instead of two
            bool inj_pending = false;                               // the last inject of a move up (level t-1 -> t, t large)
            const T* inj_src = nullptr;
            T* inj_dst = nullptr;
            struct PendingDeliver { bool on = false; const T* ec; const T* ac; T* ef; T* af; int ef_assign, af_mode; };
            std::vector<PendingDeliver> pend(s->levels + 1);
            if (t < cur) {
                // S3a deliver (interpolate + correct) level m -> m-1
                for (int m = cur; m > t; --m) {
                    Level& Lc = L[m];
                    Level& Lf = L[m - 1];
                    int ef_assign = Lf.touched ? 0 : 1;
                    if (m - 1 == t && t == 0 && ef_assign && !a_zero[m] && tiled(s, t) && (VAR ? (s->fuse_first_var || use_kvisit) : s->fuse_first) &&
                        !(use_kvisit && mid_l0)) {
                        fuse_first = true;                   // S3a of this hop happens inside the first sweep
                        fuse_ec = rotp<T>(Lc, Lc.e);
                        Lf.touched = true;
                        a_zero[m] = 1;
                        break;
                    }
                    int af_mode = (m - 1 >= 1) ? (a_zero[m - 1] ? 2 : 1) : 0;
                    const T* ac = a_zero[m] ? nullptr : (const T*)Lc.a;
                    if (af_mode == 2 && !ac) af_mode = 0;          // 0 + 0: a stays "known zero"
                    const int tag = small(m - 1) ? TAG_COARSE : (m - 1 == 0 ? TAG_DELIVER0 : TAG_DELIVER);
                    if (small(m - 1)) {
                        CoarseOp<T> o = newop(OP_DELIVER, m - 1);
                        o.gi = Lc.g; o.p[0] = rotp<T>(Lc, Lc.e); o.p[1] = ac; o.q[0] = rotp<T>(Lf, Lf.e); o.q[1] = (T*)Lf.a;
                        o.f0 = ef_assign; o.f1 = af_mode;
                        R.push(o, Lf.n_nodes);
                    } else if (t >= 1) {
                        pend[m] = PendingDeliver{true, rotp<T>(Lc, Lc.e), ac, rotp<T>(Lf, Lf.e), (T*)Lf.a, ef_assign, af_mode};
                    } else {
                        flush();
                        if (!R.plan) klaunch(R, use_bricks(R.s, Lf.g) ? k_deliver_b<T, ND> : k_deliver_v<T, ND>, use_bricks(R.s, Lf.g) ? grdb<T, ND>(Lf.g) : grdv<T>(Lf.g), blk(), 0, Lf.g, Lc.g, rotp<T>(Lc, Lc.e), ac,
                                                                                    rotp<T>(Lf, Lf.e), (T*)Lf.a, ef_assign, af_mode);
                        R.check(tag);
                    }
                    R.acct(m, ac ? 2.0 : 1.0, tag);
                    R.acct(m - 1, (ef_assign ? 1.0 : 2.0) + (af_mode == 1 ? 2.0 : af_mode == 2 ? 1.0 : 0.0), tag);
                    Lf.touched = true;
                    if (af_mode) a_zero[m - 1] = 0;
                    a_zero[m] = 1;                                  // a_m delivered
                }
            } else if (t > cur) {
                // S3b inject level m-1 -> m (same memory cells in the paper's single array)
                for (int m = cur + 1; m <= t; ++m) {
                    const int tag = small(m) ? TAG_COARSE : TAG_INJECT;
                    if (small(m)) {
                        CoarseOp<T> o = newop(OP_INJECT, m);
                        o.gi = L[m - 1].g; o.p[0] = rotp<T>(L[m - 1], L[m - 1].e); o.q[0] = rotp<T>(L[m], L[m].e);
                        R.push(o, L[m].n_nodes);
                    } else if (m == t) {
                        inj_pending = true;                         // launched together with k_d0_up below (k_rise)
                        inj_src = rotp<T>(L[m - 1], L[m - 1].e); inj_dst = rotp<T>(L[m], L[m].e);
                    } else {
                        flush();
                        if (!R.plan) klaunch(R, k_inject<T, ND>, grd(L[m].g), blk(), 0, L[m].g, L[m - 1].g, rotp<T>(L[m - 1], L[m - 1].e),
                                                                                     rotp<T>(L[m], L[m].e));
                        R.check(tag);
                    }
                    R.acct(m, 2.0, tag);
                    L[m].touched = true;
                }
            }
            // S3c carried variation d0 on level t (not needed on level 0: a_0 does not exist)
            if (t >= 1) {
                Level& Lv = L[cur];
                const T* X = rotp<T>(Lv, Lv.vk);
                const T* Y = rotp<T>(Lv, Lv.vkm1);
                if (t >= cur) {
                    const int tag = small(t) ? TAG_COARSE : TAG_D0;
                    if (small(t)) {
                        CoarseOp<T> o = newop(OP_D0_UP, t);
                        o.gi = Lv.g; o.s = 1 << (t - cur); o.p[0] = X; o.p[1] = Y; o.q[0] = (T*)Lt.d0;
                        R.push(o, Lt.n_nodes);
                    } else if (inj_pending) {
                        flush();
                        if (!R.plan) klaunch(R, k_rise<T, ND>, grd(Lt.g), blk(), 0, Lt.g, L[t - 1].g, inj_src, inj_dst, Lv.g, 1 << (t - cur),
                                             X, Y, (T*)Lt.d0);
                        R.check(TAG_INJECT);
                        inj_pending = false;
                    } else {
                        flush();
                        if (!R.plan) klaunch(R, k_d0_up<T, ND>, grd(Lt.g), blk(), 0, Lt.g, Lv.g, 1 << (t - cur), X, Y, (T*)Lt.d0);
                        R.check(tag);
                    }
                    R.acct(t, 3.0, tag);
                } else {
                    const T* A = dp_is_d0[cur] ? (const T*)Lv.d0 : rotp<T>(Lv, Lv.vkm1);
                    const T* B = dp_is_d0[cur] ? nullptr : rotp<T>(Lv, Lv.vkm2);
                    for (int m = cur; m > t; --m) {
                        bool last = (m - 1 == t);
                        T* out = last ? (T*)Lt.d0 : (T*)L[m - 1].tmp;
                        const int tag = small(m - 1) ? TAG_COARSE : TAG_D0;
                        if (small(m - 1)) {
                            CoarseOp<T> o = newop(OP_D0_DOWN, m - 1);
                            o.gi = L[m].g; o.gv = Lv.g; o.s = last ? (1 << (cur - t)) : 0;
                            o.p[0] = A; o.p[1] = B; o.p[2] = X; o.p[3] = Y; o.q[0] = out;
                            R.push(o, L[m - 1].n_nodes);
                        } else if (pend[m].on) {
                            flush();
                            const PendingDeliver& pd = pend[m];
                            if (!R.plan) klaunch(R, use_bricks(R.s, L[m - 1].g) ? k_arrive_b<T, ND> : k_arrive_v<T, ND>, use_bricks(R.s, L[m - 1].g) ? grdb<T, ND>(L[m - 1].g) : grdv<T>(L[m - 1].g), blk(), 0, L[m - 1].g, L[m].g, pd.ec, pd.ac, pd.ef,
                                                 pd.af, pd.ef_assign, pd.af_mode, A, B, out, last ? (1 << (cur - t)) : 0,
                                                 last ? cur - t : 0, Lv.g, X, Y);
                            R.check(TAG_DELIVER);
                        } else {
                            flush();
                            if (!R.plan) klaunch(R, use_bricks(R.s, L[m - 1].g) ? k_d0_down_b<T, ND> : k_d0_down_v<T, ND>, use_bricks(R.s, L[m - 1].g) ? grdb<T, ND>(L[m - 1].g) : grdv<T>(L[m - 1].g), blk(), 0, L[m - 1].g, L[m].g, A, B, out,
                                                                                                last ? (1 << (cur - t)) : 0, last ? cur - t : 0, Lv.g, X, Y);
                            R.check(tag);
                        }
                        R.acct(m, B ? 2.0 : 1.0, tag); R.acct(m - 1, 1.0, tag);
                        A = out; B = nullptr;
                    }
                }
                have_d0 = true;
            }
        }
        if (t >= 1 && !have_d0 && eta == 1) {        // first visit with eta = 1: its dp is d0 = 0
            if (small(t)) {
                CoarseOp<T> o = newop(OP_ZERO, t);
                o.count = (long long)Lt.n_alloc; o.q[0] = (T*)Lt.d0;
                R.push(o, Lt.n_nodes);
            } else {
                flush();
                if (!R.plan) R.note(cudaMemsetAsync(Lt.d0, 0, Lt.n_alloc * sizeof(T), R.st));
                R.check(TAG_OTHER);
            }
            have_d0 = true;
        }
        // K_visit: the whole visit (or, on level 0, chunks of up to 4 sweeps) in one pass over HBM
        const int maxns = kv_maxns;
        if (use_kvisit) {
            flush();
            const int v0i = Lt.e;
            int in = v0i, i1 = -1, i2 = -1, done = 0;           // rot indices of v^k, v^{k-1}, v^{k-2}
            bool interp = fuse_first;
            while (done < eta) {
                const int rem = eta - done;
                const int ns = rem >= maxns ? maxns : rem;
                const bool lastc = done + ns == eta;
                const bool addu = lastc && vi == nv - 1 && t == 0;
                const bool book = lastc && t >= 1;
                if (ns == 1) {                                   // a single trailing sweep (level 0 only)
                    int out = -1;
                    for (int b = 0; b < Lt.nrot; ++b) if (b != in) { out = b; break; }
                    if (!R.plan) launch_relax<T, ND, VAR>(R, t, rotp<T>(Lt, in), rotp<T>(Lt, out), nullptr, 0, nullptr, nullptr, addu ? (T*)s->u : nullptr);
                    R.check(addu ? TAG_RELAX0_LAST : TAG_RELAX0);
                    R.acct(t, 3.0 + (addu ? 1.0 : 0.0));
                    i2 = i1; i1 = in; in = out; done += 1;
                    continue;
                }
                int ob[3] = {-1, -1, -1}, nb = 0;               // free buffers: not the input, not v^0 (t >= 1)
                for (int b = 0; b < Lt.nrot && nb < 3; ++b)
                    if (b != in && !(t >= 1 && b == v0i)) ob[nb++] = b;
                const int b0 = ob[0], b1 = (t >= 1 || (mid_l0 && lastc)) ? ob[1] : -1, b2 = (t >= 1 && ns >= 3) ? ob[2] : -1;
                T* o0 = addu ? nullptr : rotp<T>(Lt, b0);
                const int tag = t == 0 ? TAG_VISIT0 : TAG_VISIT;
                if (!R.plan) {
                    if (interp)
                        launch_visit_ns<T, ND, true, VAR>(R, ns, t, nullptr, fuse_ec, (const T*)L[t + 1].a, o0, rotp<T>(Lt, b1), rotp<T>(Lt, b2),
                                                  nullptr, 0, nullptr, nullptr, addu ? (T*)s->u : nullptr);
                    else
                        launch_visit_ns<T, ND, false, VAR>(R, ns, t, rotp<T>(Lt, in), nullptr, nullptr, o0, rotp<T>(Lt, b1), rotp<T>(Lt, b2),
                                                   book ? (T*)Lt.a : nullptr, a_zero[t] ? 1 : 0, (book && have_d0) ? (const T*)Lt.d0 : nullptr,
                                                   rotp<T>(Lt, v0i), addu ? (T*)s->u : nullptr);
                }
                R.check(tag);
                if (interp) R.acct(t + 1, 2.0, tag);
                {
                    // compulsory passes of the fused launch vs the per-sweep figures of SURVEY 8(d)
                    const double bk = book ? (a_zero[t] ? 1.0 : 2.0) + (have_d0 ? 1.0 : 0.0) : 0.0;
                    const double comp = (interp ? 0.0 : 1.0) + 1.0 + (o0 ? 1.0 : 0.0) + (b1 >= 0 ? 1.0 : 0.0) +
                                        (b2 >= 0 ? 1.0 : 0.0) + bk + (addu ? 2.0 : 0.0);
                    const double alg = (interp ? 2.0 : 3.0) + 3.0 * (ns - 1) + (addu ? 1.0 : 0.0) + bk + (book ? 1.0 : 0.0);
                    R.acct2(t, alg + (VAR ? 3.0 * ns : 0.0), comp + (VAR ? 4.0 : 0.0), tag);   // + the three face arrays (+ omega/D in the fused form)
                }
                // rot indices of the last three iterates
                if (ns >= 3) { i2 = b2; i1 = b1; }
                else { i2 = in; i1 = b1; }                        // ns == 2: v^{k-2} is this chunk's input
                in = b0;
                interp = false;
                done += ns;
            }
            if (t >= 1) a_zero[t] = 0;
            Lt.vk = in; Lt.vkm1 = i1; Lt.vkm2 = i2; Lt.e = in; Lt.eta_last = eta;
            dp_is_d0[t] = false;
            cur = t;
            continue;
        }
        // S3d eta damped-Jacobi sweeps; S3e bookkeeping fused into the last one; S4 u += e fused
        // into the last sweep of the cycle.
        const int v0 = Lt.e;
        int in = v0, prev_in = -1, prev2 = -1;
        // a small level whose compact arrays fit in one CTA's shared memory: the whole visit is ONE record
        // of the coarse program (OP_RELAXN), the iterate stays in shared memory between the sweeps
        if (small(t) && eta >= 2 && s->coarse_relaxn &&
            3 * size_t(Lt.n_nodes) * sizeof(T) <= size_t(kRelaxnSmemMax)) {
            std::vector<int> outs(eta);
            for (int it = 0; it < eta; ++it) {
                int out = -1;
                for (int b = 0; b < Lt.nrot; ++b)
                    if (b != in && b != prev_in && !(t >= 1 && b == v0)) { out = b; break; }
                outs[it] = out;
                prev2 = prev_in; prev_in = in; in = out;
            }
            const bool book = t >= 1, addu = vi == nv - 1;
            CoarseOp<T> o = newop(OP_RELAXN, t);
            o.cf = make_coef<T>(s, t);
            o.s = eta;
            o.p[0] = rotp<T>(Lt, v0); o.p[1] = (const T*)Lt.gsrc; o.p[2] = nullptr; o.kf = faces<T>(Lt);
            o.p[3] = have_d0 ? (const T*)Lt.d0 : nullptr; o.p[4] = rotp<T>(Lt, v0);
            o.q[0] = rotp<T>(Lt, outs[eta - 1]); o.q[1] = book ? (T*)Lt.a : nullptr; o.q[2] = addu ? (T*)s->u : nullptr;
            o.qx[0] = rotp<T>(Lt, outs[eta - 2]);
            o.qx[1] = eta >= 3 ? rotp<T>(Lt, outs[eta - 3]) : nullptr;
            o.f0 = a_zero[t] ? 1 : 0;
            R.push(o, 1);                                    // act = 1: worked by one CTA
            if (Lt.n_nodes > R.run_maxnodes) R.run_maxnodes = Lt.n_nodes;
            R.acct(t, 3.0 * eta + (VAR ? 3.0 * eta : 0.0) + (book ? (a_zero[t] ? 1.0 : 2.0) + (have_d0 ? 1.0 : 0.0) + 1.0 : 0.0) +
                          (addu ? 2.0 : 0.0), TAG_COARSE);
            if (t >= 1) a_zero[t] = 0;
            Lt.vk = in; Lt.vkm1 = prev_in; Lt.vkm2 = prev2; Lt.e = in; Lt.eta_last = eta;
            dp_is_d0[t] = false;
            cur = t;
            continue;
        }
        for (int it = 0; it < eta; ++it) {
            int out = -1;
            for (int b = 0; b < Lt.nrot; ++b)
                if (b != in && b != prev_in && !(t >= 1 && b == v0)) { out = b; break; }
            bool last = (it == eta - 1);
            bool book = last && t >= 1;
            bool addu = last && vi == nv - 1;
            const int tag = small(t) ? TAG_COARSE : (t != 0 ? TAG_RELAX : (fuse_first && it == 0) ? TAG_RELAX0_FIRST : addu ? TAG_RELAX0_LAST : TAG_RELAX0);
            if (fuse_first && it == 0) {
                flush();
                if (!R.plan) launch_relax_first<T, ND, VAR>(R, t, fuse_ec, (const T*)L[t + 1].a, rotp<T>(Lt, out), addu ? (T*)s->u : nullptr);
                R.check(tag);
                R.acct(t + 1, 2.0, tag);
                R.acct(t, 2.0 + (VAR ? 3.0 : 0.0) + (addu ? 1.0 : 0.0), tag);
                prev2 = prev_in; prev_in = in; in = out;
                continue;
            }
            if (small(t)) {
                CoarseOp<T> o = newop(OP_RELAX, t);
                o.cf = make_coef<T>(s, t);
                o.p[0] = rotp<T>(Lt, in); o.p[1] = (const T*)Lt.gsrc; o.p[2] = nullptr; o.kf = faces<T>(Lt);
                o.p[3] = have_d0 ? (const T*)Lt.d0 : nullptr; o.p[4] = rotp<T>(Lt, v0);
                o.q[0] = rotp<T>(Lt, out); o.q[1] = book ? (T*)Lt.a : nullptr; o.q[2] = addu ? (T*)s->u : nullptr;
                o.f0 = a_zero[t] ? 1 : 0;
                R.push(o, Lt.n_nodes);
            } else {
                flush();
                if (!R.plan)
                    launch_relax<T, ND, VAR>(R, t, rotp<T>(Lt, in), rotp<T>(Lt, out), book ? (T*)Lt.a : nullptr, a_zero[t] ? 1 : 0,
                                             have_d0 ? (const T*)Lt.d0 : nullptr, rotp<T>(Lt, v0), addu ? (T*)s->u : nullptr);
                R.check(tag);
            }
            R.acct(t, 3.0 + (VAR ? 3.0 : 0.0) + (book ? (a_zero[t] ? 1.0 : 2.0) + (have_d0 ? 1.0 : 0.0) + (eta > 1 ? 1.0 : 0.0) : 0.0) +
                          (addu ? (tiled(s, t) && t == 0 ? 1.0 : 2.0) : 0.0), tag);
            prev2 = prev_in; prev_in = in; in = out;
        }
        if (t >= 1) a_zero[t] = 0;
        Lt.vk = in; Lt.vkm1 = prev_in; Lt.vkm2 = prev2; Lt.e = in; Lt.eta_last = eta;
        dp_is_d0[t] = (eta == 1);
        cur = t;
    }
    flush();
    if (R.s1_at_end) rec_norm<T, ND, VAR>(R, true, true, true);    // S1 + S5 of the new u: the loop condition
}

// ---------------------------------------------------------------------------------------------
// Classic V(eta1, eta2) cycle on the same hierarchy and kernels:
// (a) eta1 sweeps, (b) r = g - A v restricted by full weighting, (c) exact solve on the coarsest
// level (one interior node), (d) v += S^ e, (e) eta2 sweeps.  Level 0 works on u itself with g = f.
// ---------------------------------------------------------------------------------------------
// n sweeps on level m starting from `cur`; the last one writes into `final_dst` when given and
// possible.  Returns the array that holds the result.
template <class T, int ND, bool VAR>
T* v_sweeps(Rec& R, int m, T* cur, int n, T* final_dst) {
    homg_solver* s = R.s;
    Level& Lm = s->L[m];
    auto pick = [&](const T* not1, const T* not2) -> T* {
        for (int b = 0; b < Lm.nrot; ++b) {
            T* c = rotp<T>(Lm, b);
            if (c != not1 && c != not2) return c;
        }
        return nullptr;
    };
    const int maxns = std::min(s->fuse_visit, 4);
    int done = 0;
    while (done < n) {
        const int rem = n - done;
        const bool fuse = !VAR && maxns >= 2 && tiled(s, m) && rem >= 2;
        const int ns = fuse ? std::min(rem, maxns) : 1;
        const bool lastc = done + ns == n;
        T* out = (lastc && final_dst && final_dst != cur) ? final_dst : pick(cur, final_dst);
        if (fuse) {
            launch_visit_ns<T, ND, false>(R, ns, m, cur, nullptr, nullptr, out, nullptr, nullptr, nullptr, 0, nullptr, nullptr, nullptr);
            R.check(m == 0 ? TAG_VISIT0 : TAG_VISIT);
            R.acct2(m, 3.0 * ns, 3.0, m == 0 ? TAG_VISIT0 : TAG_VISIT);
        } else {
            launch_relax<T, ND, VAR>(R, m, cur, out, nullptr, 0, nullptr, nullptr, nullptr);
            R.check(m == 0 ? TAG_RELAX0 : TAG_RELAX);
            R.acct(m, 3.0 + (VAR ? 3.0 : 0.0), m == 0 ? TAG_RELAX0 : TAG_RELAX);
        }
        cur = out;
        done += ns;
    }
    return cur;
}

template <class T, int ND, bool VAR>
void rec_vcycle(Rec& R) {
    homg_solver* s = R.s;
    const int M = s->levels - 1;
    std::vector<Level>& L = s->L;
    // norm of the current u -> history (the classic cycle has no residual of the iterate it starts from)
    rec_norm<T, ND, VAR>(R, false, true, false);
    std::vector<T*> cur(s->levels, nullptr);
    cur[0] = (T*)s->u;
    for (int m = 0; m < M; ++m) {
        Level& Lm = L[m];
        if (m >= 1) {                                            // e_m = 0
            cur[m] = rotp<T>(Lm, 0);
            R.note(cudaMemsetAsync(cur[m], 0, Lm.n_alloc * sizeof(T), R.st));
            R.check(TAG_OTHER);
        }
        R.g_override = m == 0 ? s->f : nullptr;
        cur[m] = v_sweeps<T, ND, VAR>(R, m, cur[m], s->v_eta1, nullptr);                       // (a)
        R.g_override = nullptr;
        if (m == 0) {                                            // (b) K_res: r -> g_0 scratch, g_1 = P r
            R.u_override = cur[0];
            const bool have_g1 = rec_norm<T, ND, VAR>(R, true, false, true);
            R.u_override = nullptr;
            if (!have_g1) {
                klaunch(R, k_restrict<T, ND>, grd(L[1].g), blk(), 0, L[1].g, L[0].g, (const T*)L[0].gsrc, (T*)L[1].gsrc);
                R.check(TAG_RESTRICT);
                R.acct(0, 1.0, TAG_RESTRICT); R.acct(1, 1.0, TAG_RESTRICT);
            }
        } else {
            klaunch(R, k_residual<T, ND, VAR>, grd(Lm.g), blk(), 0, Lm.g, make_coef<T>(s, m), (const T*)cur[m],
                    (const T*)Lm.gsrc, faces<T>(Lm), (T*)Lm.tmp, s->partial);
            R.check(TAG_OTHER);
            R.acct(m, 3.0 + (VAR ? 3.0 : 0.0), TAG_OTHER);
            klaunch(R, k_restrict<T, ND>, grd(L[m + 1].g), blk(), 0, L[m + 1].g, Lm.g, (const T*)Lm.tmp, (T*)L[m + 1].gsrc);
            R.check(TAG_RESTRICT);
            R.acct(m, 1.0, TAG_RESTRICT); R.acct(m + 1, 1.0, TAG_RESTRICT);
        }
    }
    // (c) coarsest level: exact solve (one interior node)
    cur[M] = rotp<T>(L[M], 0);
    if (M >= 1) {
        R.note(cudaMemsetAsync(cur[M], 0, L[M].n_alloc * sizeof(T), R.st));
        R.check(TAG_OTHER);
        klaunch(R, k_coarsest_solve<T, ND, VAR>, dim3(1), dim3(32), 0, L[M].g, make_coef<T>(s, M), (const T*)L[M].gsrc,
                faces<T>(L[M]), cur[M]);
        R.check(TAG_COARSE);
    }
    for (int m = M - 1; m >= 0; --m) {
        Level& Lm = L[m];
        klaunch(R, use_bricks(R.s, Lm.g) ? k_prolong_add_b<T, ND> : k_prolong_add_v<T, ND>, use_bricks(R.s, Lm.g) ? grdb<T, ND>(Lm.g) : grdv<T>(Lm.g), blk(), 0, Lm.g, L[m + 1].g, (const T*)cur[m + 1], cur[m]);   // (d)
        R.check(m == 0 ? TAG_DELIVER0 : TAG_DELIVER);
        R.acct(m, 2.0, m == 0 ? TAG_DELIVER0 : TAG_DELIVER); R.acct(m + 1, 1.0, m == 0 ? TAG_DELIVER0 : TAG_DELIVER);
        R.g_override = m == 0 ? s->f : nullptr;
        cur[m] = v_sweeps<T, ND, VAR>(R, m, cur[m], s->v_eta2, m == 0 ? (T*)s->u : nullptr);     // (e)
        R.g_override = nullptr;
    }
    if (cur[0] != (T*)s->u) {                                    // eta2 = 0, or a single sweep that started from u
        R.note(cudaMemcpyAsync(s->u, cur[0], L[0].n_alloc * sizeof(T), cudaMemcpyDeviceToDevice, R.st));
        R.check(TAG_OTHER);
        R.acct(0, 2.0, TAG_OTHER);
    }
}

// ---------------------------------------------------------------------------------------------
// Paper-literal mode: Algorithm L on the GPU — one fine-grid array, one whole-grid
// launch per iteration at every level.  A measured prior-art row, not the product.
// ---------------------------------------------------------------------------------------------
template <class T, int ND, bool VAR>
void rec_literal(Rec& R) {
    homg_solver* s = R.s;
    const int M = s->levels - 1;
    std::vector<Level>& L = s->L;
    Level& L0 = L[0];
    if (s->pow2) {
        // PAPER.md section 3 (homg_pow2.cuh): the residual, then nested full weighting on the four anchored lattices
        rec_norm<T, ND, VAR>(R, true, true, false);
        const int N = L0.g.nx;
        auto srcs = [&](int m) { P2Src<T> q; for (int a = 0; a < 4; ++a) q.p[a] = (const T*)s->p2src[a][m]; return q; };
        auto dsts = [&](int m) { P2Dst<T> q; for (int a = 0; a < 4; ++a) q.p[a] = (T*)s->p2src[a][m]; return q; };
        for (int m = 1; m <= M; ++m) {
            const LevelGeom& gc = L[m].g;
            const dim3 grid((gc.nx + 31) / 32, (gc.ny + 7) / 8, 4);
            klaunch(R, k_p2_restrict<T>, grid, blk(), 0, gc, L[m - 1].g, N, m == 1 ? 1 : 0, (const T*)L0.gsrc, srcs(m == 1 ? 1 : m - 1),
                    dsts(m));
            R.check(TAG_RESTRICT);
            R.acct(m - 1, m == 1 ? 4.0 : 4.0, TAG_RESTRICT); R.acct(m, 4.0, TAG_RESTRICT);
        }
        int ic = 0, ip = 1, in = 2;
        R.note(cudaMemsetAsync(L0.rot[ic], 0, L0.n_alloc * sizeof(T), R.st)); R.check(TAG_OTHER);
        R.note(cudaMemsetAsync(L0.rot[ip], 0, L0.n_alloc * sizeof(T), R.st)); R.check(TAG_OTHER);
        R.acct(0, 2.0, TAG_OTHER);
        for (size_t vi = 0; vi < s->sched_lv.size(); ++vi) {
            const int m = s->sched_lv[vi];
            for (int it = 0; it < s->sched_it[vi]; ++it) {
                klaunch(R, k_iter_p2<T>, grd(L0.g), blk(), 0, L0.g, L[m].g, N, m, make_coef<T>(s, m), (const T*)L0.rot[ic],
                        (const T*)L0.rot[ip], (T*)L0.rot[in], (const T*)L0.gsrc, srcs(m == 0 ? 1 : m));
                R.check(m == 0 ? TAG_RELAX0 : TAG_RELAX);
                R.acct(0, 3.0, m == 0 ? TAG_RELAX0 : TAG_RELAX);
                const int t = ip; ip = ic; ic = in; in = t;
            }
        }
        const long long n16 = (long long)(L0.n_alloc * sizeof(T) / 16);
        klaunch(R, k_add_v<T>, dim3((unsigned)((n16 + 255) / 256)), dim3(256), 0, (T*)s->u, (const T*)L0.rot[ic], n16);
        R.check(TAG_OTHER);
        R.acct(0, 3.0, TAG_OTHER);
        return;
    }
    const bool have_g1 = rec_norm<T, ND, VAR>(R, true, true, true);           // r -> g_0, norm, g_1
    for (int m = have_g1 ? 2 : 1; m <= M; ++m) {
        klaunch(R, k_restrict<T, ND>, grd(L[m].g), blk(), 0, L[m].g, L[m - 1].g, (const T*)L[m - 1].gsrc, (T*)L[m].gsrc);
        R.check(TAG_RESTRICT);
        R.acct(m - 1, 1.0, TAG_RESTRICT); R.acct(m, 1.0, TAG_RESTRICT);
    }
    int ic = 0, ip = 1, in = 2;                                                // cur, prev, nxt among the 3 level-0 buffers
    R.note(cudaMemsetAsync(L0.rot[ic], 0, L0.n_alloc * sizeof(T), R.st)); R.check(TAG_OTHER);
    R.note(cudaMemsetAsync(L0.rot[ip], 0, L0.n_alloc * sizeof(T), R.st)); R.check(TAG_OTHER);
    R.acct(0, 2.0, TAG_OTHER);
    for (size_t vi = 0; vi < s->sched_lv.size(); ++vi) {
        const int m = s->sched_lv[vi];
        for (int it = 0; it < s->sched_it[vi]; ++it) {
            klaunch(R, k_iter_literal<T, ND, VAR>, grd(L0.g), blk(), 0, L0.g, L[m].g, m, make_coef<T>(s, m),
                    (const T*)L0.rot[ic], (const T*)L0.rot[ip], (T*)L0.rot[in], (const T*)L[m].gsrc, faces<T>(L[m]));
            R.check(m == 0 ? TAG_RELAX0 : TAG_RELAX);
            R.acct(0, 3.0, m == 0 ? TAG_RELAX0 : TAG_RELAX);                   // 1 WU: read cur, prev; write nxt
            const int t = ip; ip = ic; ic = in; in = t;
        }
    }
    const long long n16 = (long long)(L0.n_alloc * sizeof(T) / 16);
    klaunch(R, k_add_v<T>, dim3((unsigned)((n16 + 255) / 256)), dim3(256), 0, (T*)s->u, (const T*)L0.rot[ic], n16);
    R.check(TAG_OTHER);
    R.acct(0, 3.0, TAG_OTHER);
}

template <class T, int ND, bool VAR>
void rec_sample(Rec& R) {
    homg_solver* s = R.s;
    for (int m = 1; m < s->levels; ++m) {
        klaunch(R, k_sample_coef<T, ND>, grd(s->L[m].g), blk(), 0, s->L[m].g, s->L[m - 1].g, (const T*)s->L[m - 1].k,
                                                                   (T*)s->L[m].k);
        R.check(TAG_OTHER);
    }
    for (int m = 0; m < s->levels; ++m) {               // S0: face coefficients of every level
        Level& Lm = s->L[m];
        klaunch(R, k_faces<T, ND>, grd(Lm.g), blk(), 0, Lm.g, (const T*)Lm.k, (T*)Lm.fz, (T*)Lm.fy, (T*)Lm.fx);
        R.check(TAG_OTHER);
        if (Lm.wd) {
            klaunch(R, k_wdiag<T, ND>, grd(Lm.g), blk(), 0, Lm.g, make_coef<T>(s, m), faces<T>(Lm), (T*)Lm.wd);
            R.check(TAG_OTHER);
        }
    }
}

template <class T, int ND>
void rec_pack(Rec& R, const void* dense, void* padded, int zero_boundary) {
    const LevelGeom& g = R.s->L[0].g;
    klaunch(R, k_pack<T, ND>, grd(g), blk(), 0, g, (const T*)dense, (T*)padded, zero_boundary);
    R.check(TAG_OTHER);
}

template <class T, int ND>
void rec_unpack(Rec& R, const void* padded, void* dense) {
    const LevelGeom& g = R.s->L[0].g;
    klaunch(R, k_unpack<T, ND>, grd(g), blk(), 0, g, (const T*)padded, (T*)dense);
    R.check(TAG_OTHER);
}

// dispatch on (dtype, ndim, var)
#define HOMG_DISPATCH(s, FN, ...)                                                            \
    do {                                                                                     \
        if ((s)->dtype == HOMG_F32) {                                                        \
            if ((s)->ndim == 2) FN<float, 2, false>(__VA_ARGS__);                            \
            else if ((s)->var) FN<float, 3, true>(__VA_ARGS__);                              \
            else FN<float, 3, false>(__VA_ARGS__);                                           \
        } else {                                                                             \
            if ((s)->ndim == 2) FN<double, 2, false>(__VA_ARGS__);                           \
            else if ((s)->var) FN<double, 3, true>(__VA_ARGS__);                             \
            else FN<double, 3, false>(__VA_ARGS__);                                          \
        }                                                                                    \
    } while (0)

#define HOMG_DISPATCH2(s, FN, ...)                                                           \
    do {                                                                                     \
        if ((s)->dtype == HOMG_F32) {                                                        \
            if ((s)->ndim == 2) FN<float, 2>(__VA_ARGS__); else FN<float, 3>(__VA_ARGS__);   \
        } else {                                                                             \
            if ((s)->ndim == 2) FN<double, 2>(__VA_ARGS__); else FN<double, 3>(__VA_ARGS__); \
        }                                                                                    \
    } while (0)


template <class T, int ND, bool VAR>
cudaError_t set_attr() {
    cudaError_t e = cudaFuncSetAttribute(k_relax_tma<T, ND, VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         relax_smem_bytes<T, ND, VAR>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_relax_first<T, ND, VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             first_smem_bytes<T, ND, VAR>());
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_res_tma<T, ND, VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                res_smem_bytes<T, ND, VAR>());
}

template <class T, int ND, bool VAR>
cudaError_t set_attr_coarse() {
    cudaError_t e = cudaFuncSetAttribute(k_coarse_run<T, ND, VAR, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRelaxnSmemMax);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_coarse_run<T, ND, VAR, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRelaxnSmemMax);
}

template <class T, int ND, int NS>
cudaError_t set_attr_visit1() {
    cudaError_t e = cudaFuncSetAttribute(k_visit<T, ND, NS, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         visit_smem_bytes<T, ND, NS, false>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_visit<T, ND, NS, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             visit_smem_bytes<T, ND, NS, false>());
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_visit<T, ND, NS, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                visit_smem_bytes<T, ND, NS, true>());
}
template <class T, int NS>
cudaError_t set_attr_visit() {
    cudaError_t e = set_attr_visit1<T, 2, NS>();
    if (e != cudaSuccess) return e;
    if ((e = set_attr_visit1<T, 3, NS>()) != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_visit3<T, NS, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, visit3_smem_bytes<T, NS, false, false>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_visit3<T, NS, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, visit3_smem_bytes<T, NS, false, true>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_visit3<T, NS, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, visit3_smem_bytes<T, NS, true, false>());
    if (e != cudaSuccess || NS != 2) return e;
    e = cudaFuncSetAttribute(k_visit3<T, 2, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, visit3_smem_bytes<T, 2, false, false, true>());
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_visit3<T, 2, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, visit3_smem_bytes<T, 2, true, false, true>());
}

}  // namespace

cudaError_t exec_init(homg_solver* s) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&s->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
    if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) return e != cudaSuccess ? e : cudaErrorNotSupported;
    s->encode_tiled = fn;
    if ((e = set_attr<float, 2, false>()) != cudaSuccess) return e;
    if ((e = set_attr<float, 3, false>()) != cudaSuccess) return e;
    if ((e = set_attr<float, 3, true>()) != cudaSuccess) return e;
    if ((e = set_attr<double, 2, false>()) != cudaSuccess) return e;
    if ((e = set_attr<double, 3, false>()) != cudaSuccess) return e;
    if ((e = set_attr<double, 3, true>()) != cudaSuccess) return e;
    if ((e = set_attr_coarse<float, 2, false>()) != cudaSuccess) return e;
    if ((e = set_attr_coarse<float, 3, false>()) != cudaSuccess) return e;
    if ((e = set_attr_coarse<float, 3, true>()) != cudaSuccess) return e;
    if ((e = set_attr_coarse<double, 2, false>()) != cudaSuccess) return e;
    if ((e = set_attr_coarse<double, 3, false>()) != cudaSuccess) return e;
    if ((e = set_attr_coarse<double, 3, true>()) != cudaSuccess) return e;
    if ((e = set_attr_visit<float, 2>()) != cudaSuccess) return e;
    if ((e = set_attr_visit<float, 3>()) != cudaSuccess) return e;
    if ((e = set_attr_visit<float, 4>()) != cudaSuccess) return e;
    if ((e = set_attr_visit<double, 2>()) != cudaSuccess) return e;
    if ((e = set_attr_visit<double, 3>()) != cudaSuccess) return e;
    if ((e = set_attr_visit<double, 4>()) != cudaSuccess) return e;
    return cudaSuccess;
}

cudaError_t exec_prepare(homg_solver* s) {
    if (s->inner) return exec_prepare(s->inner);                 // the outer problem has no coarse levels
    if (s->prog_ready || s->vcycle || s->literal) return cudaSuccess;       // the V-cycle has no coarse program
    Rec P{s, s->stream};
    P.plan = true;
    P.skip_s1 = s->given_g0;
    HOMG_DISPATCH(s, rec_cycle, P);
    if (P.err != cudaSuccess) return P.err;
    if (!P.prog.empty()) {
        cudaError_t e = cudaMalloc(&s->prog_dev, P.prog.size());
        if (e != cudaSuccess) { s->prog_dev = nullptr; return e; }
        e = cudaMemcpy(s->prog_dev, P.prog.data(), P.prog.size(), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { cudaFree(s->prog_dev); s->prog_dev = nullptr; return e; }
    }
    s->prog_ready = true;
    return cudaSuccess;
}

// Mixed-precision outer cycle (the restart is a defect-correction loop):
// `s` is the fp64 outer problem (one level: u, f, r), s->inner the fp32 hierarchy.  r = f - A u and its norm
// in fp64 (K_res), r rounded to fp32 = the inner right-hand side, ONE fp32 HOMG cycle from e = 0, u += e in fp64.
// cond != 0: the loop body of homg_solve — the fp64 residual and its norm come LAST (of the new u) and set the loop
// condition; the first kernel of the body carries no PDL attribute (see Rec)
template <int ND>
cudaError_t cycle_mixed(homg_solver* s, cudaStream_t st, unsigned long long cond = 0) {
    homg_solver* in = s->inner;
    Rec R{s, st};
    auto outer_norm = [&]() {
        if (s->var) rec_norm<double, ND, true>(R, true, true, false);
        else rec_norm<double, ND, false>(R, true, true, false);
    };
    if (!cond) outer_norm();
    else R.nopdl_next = true;
    const LevelGeom& go = s->L[0].g;
    const LevelGeom& gi = in->L[0].g;
    // g_0 of the inner hierarchy = fl32(r): the inner cycle's own S1 would compute f_in - A 0 = f_in, so it is skipped
    const dim3 g4((go.nx + 127) / 128, (go.ny + 7) / 8, go.nz);
    klaunch(R, k_cvt4<ND, false>, g4, blk(), 0, go, gi, (double*)s->L[0].gsrc, (float*)in->L[0].gsrc);
    R.check(TAG_OTHER);
    R.acct(0, 1.5, TAG_OTHER);
    R.note(cudaMemsetAsync(in->u, 0, in->L[0].n_alloc * sizeof(float), st));
    R.check(TAG_OTHER);
    R.acct(0, 0.5, TAG_OTHER);
    Rec Ri{in, st};
    Ri.skip_s1 = in->given_g0;
    HOMG_DISPATCH(in, rec_cycle, Ri);
    klaunch(R, k_cvt4<ND, true>, g4, blk(), 0, go, gi, (double*)s->u, (float*)in->u);
    R.check(TAG_OTHER);
    R.acct(0, 2.5, TAG_OTHER);
    if (cond) { R.cond = cond; outer_norm(); }
    s->launches_per_cycle = R.launches + Ri.launches;
    s->bytes_cycle_all = R.bytes_all + Ri.bytes_all;
    s->bytes_cycle_l0 = R.bytes_l0 + Ri.bytes_l0;
    for (int t = 0; t < TAG_COUNT; ++t) s->comp_by_tag[t] = R.comp_tag[t] + Ri.comp_tag[t];
    return R.err != cudaSuccess ? R.err : Ri.err;
}

cudaError_t exec_cvt_coef_to_inner(homg_solver* s, cudaStream_t st) {
    homg_solver* in = s->inner;
    Rec R{s, st};
    klaunch(R, k_cvt_pad<float, double, 3, false>, grd(in->L[0].g), blk(), 0, in->L[0].g, s->L[0].g, (const double*)s->L[0].k,
            (float*)in->L[0].k);
    R.check(TAG_OTHER);
    return R.err;
}

cudaError_t exec_cycle(homg_solver* s, cudaStream_t st) {
    if (s->inner) return s->ndim == 2 ? cycle_mixed<2>(s, st) : cycle_mixed<3>(s, st);
    Rec R{s, st};
    if (s->vcycle) HOMG_DISPATCH(s, rec_vcycle, R);
    else if (s->literal) HOMG_DISPATCH(s, rec_literal, R);
    else HOMG_DISPATCH(s, rec_cycle, R);
    s->launches_per_cycle = R.launches;
    s->bytes_cycle_all = R.bytes_all;
    s->bytes_cycle_l0 = R.bytes_l0;
    for (int t = 0; t < TAG_COUNT; ++t) s->comp_by_tag[t] = R.comp_tag[t];
    return R.err;
}

// homg_solve, prologue: S1 of the initial guess (norm -> history, loop condition)
cudaError_t exec_solve_prologue(homg_solver* s, cudaStream_t st, unsigned long long cond) {
    Rec R{s, st};
    R.cond = cond;
    if (s->inner) {                                  // mixed precision: the fp64 residual of the outer problem (one level)
        HOMG_DISPATCH(s, rec_norm, R, true, true, false);
        return R.err;
    }
    HOMG_DISPATCH(s, rec_norm, R, true, true, true);
    return R.err;
}
// homg_solve, loop body: S2..S4 of one cycle, then S1 of the new u
cudaError_t exec_solve_body(homg_solver* s, cudaStream_t st, unsigned long long cond) {
    if (s->inner) return s->ndim == 2 ? cycle_mixed<2>(s, st, cond) : cycle_mixed<3>(s, st, cond);
    Rec R{s, st};
    R.cond = cond;
    R.s1_at_end = true;
    HOMG_DISPATCH(s, rec_cycle, R);
    s->launches_per_cycle = R.launches;
    s->bytes_cycle_all = R.bytes_all;
    s->bytes_cycle_l0 = R.bytes_l0;
    for (int t = 0; t < TAG_COUNT; ++t) s->comp_by_tag[t] = R.comp_tag[t];
    return R.err;
}

cudaError_t exec_cycle_profiled(homg_solver* s, cudaStream_t st, double* ms_by_tag, int* launches_by_tag,
                                double* bytes_by_tag) {
    std::vector<cudaEvent_t> ev;
    std::vector<int> tag;
    cudaEvent_t e0;
    cudaEventCreate(&e0);
    cudaEventRecord(e0, st);
    Rec R{s, st};
    R.ev = &ev; R.ev_tag = &tag;
    if (s->vcycle) HOMG_DISPATCH(s, rec_vcycle, R);
    else if (s->literal) HOMG_DISPATCH(s, rec_literal, R);
    else HOMG_DISPATCH(s, rec_cycle, R);
    cudaError_t e = cudaStreamSynchronize(st);
    if (R.err == cudaSuccess) R.err = e;
    cudaEvent_t prev = e0;
    for (size_t i = 0; i < ev.size(); ++i) {
        float ms = 0.f;
        if (R.err == cudaSuccess) cudaEventElapsedTime(&ms, prev, ev[i]);
        ms_by_tag[tag[i]] += double(ms);
        launches_by_tag[tag[i]] += 1;
        prev = ev[i];
    }
    for (int t = 0; t < TAG_COUNT; ++t) bytes_by_tag[t] += R.bytes_tag[t];
    cudaEventDestroy(e0);
    for (auto x : ev) cudaEventDestroy(x);
    return R.err;
}

cudaError_t exec_norm_only(homg_solver* s, cudaStream_t st) {
    Rec R{s, st};
    HOMG_DISPATCH(s, rec_norm, R, false, false, false);
    return R.err;
}

cudaError_t exec_sample_coef(homg_solver* s, cudaStream_t st) {
    Rec R{s, st};
    HOMG_DISPATCH(s, rec_sample, R);
    return R.err;
}

cudaError_t exec_pack(homg_solver* s, cudaStream_t st, const void* dense_dev, void* padded, int zero_boundary) {
    Rec R{s, st};
    HOMG_DISPATCH2(s, rec_pack, R, dense_dev, padded, zero_boundary);
    return R.err;
}

cudaError_t exec_unpack(homg_solver* s, cudaStream_t st, const void* padded, void* dense_dev) {
    Rec R{s, st};
    HOMG_DISPATCH2(s, rec_unpack, R, padded, dense_dev);
    return R.err;
}

}  // namespace homg
