// homg_internal.h — host-side structures of libhomg.so (not installed; include/homg.h is the ABI).
#pragma once
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/homg.h"
#include "homg_geom.h"

namespace homg {

constexpr int kMaxLevels = 32;
constexpr int kNumRot = 4;   // rotating correction buffers per level (v0, v^k, v^{k-1}, v^{k-2})

// One level of the hierarchy.  All pointers are carved out of
// the caller's workspace; every array holds n_alloc scalars.
struct Level {
    LevelGeom g;
    size_t n_alloc = 0;        // scalars per array (pp*nz, rounded up so that bytes % 256 == 0, + pad)
    long long n_nodes = 0;     // nx*ny*nz
    double h = 0;              // mesh width 2^m h
    void* rot[kNumRot] = {};   // correction buffers (level 0 uses 3)
    int nrot = 0;
    void* a = nullptr;         // pending increments (levels >= 1)
    void* gsrc = nullptr;      // restricted residual g_m (level 0: the residual itself)
    void* d0 = nullptr;        // carried variation (levels >= 1)
    void* tmp = nullptr;       // scratch of the d0 prolongation chain (levels >= 1)
    void* k = nullptr;         // nodal coefficient (HOMG_DIFFUSION7)
    void* fz = nullptr;        // face coefficients towards +z / +y / +x (HOMG_DIFFUSION7; homg_geom.h Faces)
    void* fy = nullptr;
    void* fx = nullptr;
    void* wd = nullptr;        // omega / D per node, D = the operator's diagonal (HOMG_DIFFUSION7; S0; read by K_visit's variable-coefficient form)
    // --- executor state while one cycle is being recorded ---
    int e = 0;                 // rot index holding the materialised correction e_m
    bool touched = false;      // e_m / a_m already defined in this cycle
    int vk = -1, vkm1 = -1, vkm2 = -1;   // rot indices of v^eta, v^{eta-1}, v^{eta-2} of the last visit
    int eta_last = 0;
};

struct Plan {                  // result of plan_layout: sizes only, no pointers
    int ndim = 0, levels = 0, esize = 0;
    bool var = false;
    bool pow2 = false;         // HOMG_POISSON5_POW2: level m >= 1 holds the four anchored source arrays only
    std::vector<LevelGeom> g;
    std::vector<size_t> n_alloc;
    size_t staging_bytes = 0;  // dense level-0 array for pack/unpack
    size_t partial_count = 0;  // doubles for per-block norm partials
    size_t total_bytes = 0;
};

bool plan_layout(int ndim, const int64_t* dims, int levels, homg_stencil st, homg_dtype dt, Plan& P,
                 std::string* why);

int build_schedule(int kind, int levels, int maxI, const int* xl, const int* xi, int xlen,
                   std::vector<int>& lv, std::vector<int>& it, std::string* why);

}  // namespace homg

struct homg_solver {
    int ndim = 0, levels = 0;
    homg_stencil stencil = HOMG_POISSON5;
    homg_dtype dtype = HOMG_F64;
    bool var = false;
    double omega = 0, h = 0;
    int max_iters = 4;
    long long coarse_threshold = 0;  // levels with <= this many nodes run inside K_coarse launches
    int coarse_cluster = 0;          // 0: automatic cluster size (1, 4 or 8 CTAs)
    void* prog_dev = nullptr;        // CoarseOp records of one cycle (library-owned device memory)
    bool prog_ready = false;
    bool coarse_relaxn = true;       // a visit of a small level = one OP_RELAXN record (HOMG_COARSE_RELAXN=0: one record per sweep)
    bool use_graph = true;
    long long tiled_min_nodes = 0;   // levels with >= this many nodes use the TMA-tiled kernels
    int march_chunk = 0;             // 0: automatic
    bool pdl = true;                 // programmatic dependent launch on every kernel (HOMG_PDL=0 disables)
    bool fuse_first = true;          // fused interpolate+correct+relax first sweep (HOMG_FUSE_FIRST=0 disables)
    bool fuse_first_var = false;     // ... for the variable-coefficient stencil: measured slower than deliver + sweep
                                     // (cfg5: 535 us vs 64 + 190 us), off unless HOMG_FUSE_FIRST_VAR=1
    bool given_g0 = false;           // this is the inner hierarchy of a mixed-precision solver: g_0 is written by the outer loop
    homg_solver* inner = nullptr;    // mixed precision: this is the fp64 outer problem (1 level), inner the
                                     // fp32 hierarchy that runs the correction cycle; owned by this object
    bool literal = false;            // paper-literal whole-grid iteration, Algorithm L
    bool pow2 = false;               // PAPER.md section 3: power-of-two grid (whole-grid iteration, homg_pow2.cuh)
    void* p2src[4][homg::kMaxLevels] = {};   // restricted sources on the four anchored lattices, levels >= 1
    bool vcycle = false;             // classic V(v_eta1, v_eta2) instead of the MFMG cycle
    int v_eta1 = 2, v_eta2 = 1;
    int fuse_visit = 4;              // K_visit: up to this many sweeps of a visit in one pass (0/1: off; HOMG_FUSE_VISIT)
    int visit3 = 2;                  // 3-D K_visit: 2 = homg_visit3.cuh for every form (default); 1 = only the level-0 / plain
                                     // forms, bookkeeping visits on homg_visit.cuh; 0 = homg_visit.cuh (the r01 kernel) throughout
    bool visit_var = true;           // K_visit for the variable-coefficient stencil: level 0, two sweeps per pass, multiplies by the
                                     // precomputed RN(omega/D) (rounding-level difference to the per-sweep kernels); HOMG_VISIT_VAR=0: per sweep
    bool bricks = true;              // level-change kernels in brick form (homg_bricks.cuh); HOMG_BRICKS=0: one pack per thread
    int sm_count = 148;
    void* encode_tiled = nullptr;    // cuTensorMapEncodeTiled, fetched from the driver at create
    std::vector<int> sched_lv, sched_it;
    std::vector<homg::Level> L;
    // level-0 extras
    void* u = nullptr;
    void* f = nullptr;
    void* staging = nullptr;
    double* partial = nullptr;   // per-block partial sums of r^2
    size_t partial_count = 0;
    double* hist = nullptr;      // device norm^2 history
    int hist_cap = 0;
    int* slot = nullptr;         // device: next history slot
    double* scalar = nullptr;    // device: result of a norm-only pass
    char* ws_base = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;       // the caller's stream: all work is issued here
    cudaStream_t cap_stream = nullptr;   // private stream used only to capture the graph
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t graph_exec = nullptr;
    cudaGraph_t solve_graph = nullptr;   // homg_solve: S1, then a WHILE node whose body is one cycle (S2..S4, S1)
    cudaGraphExec_t solve_exec = nullptr;
    cudaGraph_t solve_body = nullptr;    // the WHILE node's body (owned by solve_graph)
    int solve_census[5] = {};            // kernel / memset / memcpy / conditional / other nodes of solve_graph + body
    void* solve_params = nullptr;        // device: SolveParams (tolerance^2, last history slot)
    bool have_rhs = false, have_coef = false;
    long cycles_issued = 0;
    int launches_per_cycle = 0;
    double bytes_cycle_all = 0, bytes_cycle_l0 = 0;
    double comp_by_tag[32] = {};         // compulsory bytes of one cycle per kernel class
    std::string err;
};
