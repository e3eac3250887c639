// homg_layout.cu — hierarchy layout in HBM and the MFMG schedule table (host only).
#include <algorithm>

#include "homg_internal.h"

namespace homg {

static size_t round_up(size_t v, size_t m) { return (v + m - 1) / m * m; }

// Every level array: rows of nx nodes padded to a multiple of 128 B, ny rows per plane, nz planes,
// contiguous; the array length is rounded up to 256 B and followed by one spare padded row so that
// vectorised row loads of the last row never leave the array.          (north_star item 1)
bool plan_layout(int ndim, const int64_t* dims, int levels, homg_stencil st, homg_dtype dt, Plan& P,
                 std::string* why) {
    auto fail = [&](const char* m) { if (why) *why = m; return false; };
    if (!dims) return fail("dims is null");
    if (ndim != 2 && ndim != 3) return fail("ndim must be 2 or 3");
    if (levels < 1 || levels > kMaxLevels) return fail("levels out of range");
    if (dt != HOMG_F32 && dt != HOMG_F64) return fail("dtype must be HOMG_F32 or HOMG_F64");
    if (st == HOMG_POISSON5 && ndim != 2) return fail("HOMG_POISSON5 needs ndim = 2");
    if ((st == HOMG_POISSON7 || st == HOMG_DIFFUSION7) && ndim != 3) return fail("7-point stencils need ndim = 3");
    if (st == HOMG_POISSON5_POW2 && ndim != 2) return fail("HOMG_POISSON5_POW2 needs ndim = 2");
    if (st != HOMG_POISSON5 && st != HOMG_POISSON7 && st != HOMG_DIFFUSION7 && st != HOMG_POISSON5_POW2) return fail("unknown stencil");
    int64_t q = int64_t(1) << (levels - 1);
    const bool pow2 = st == HOMG_POISSON5_POW2;
    if (pow2) {
        // PAPER.md section 3: N = 2^k nodes per side; the coarsest lattice of a half is {anchor, central point}: l <= N/2
        const int64_t N = dims[0];
        if (dims[1] != N || N < 8 || N > (int64_t(1) << 15) || (N & (N - 1)) != 0) return fail("HOMG_POISSON5_POW2: dims = (N, N), N = 2^k, 8 <= N <= 32768");
        if (q > N / 2) return fail("HOMG_POISSON5_POW2: 2^(levels-1) must not exceed N/2");
    }
    for (int a = 0; a < ndim && !pow2; ++a) {
        if (dims[a] < 3 || dims[a] > (int64_t(1) << 30)) return fail("dims out of range");
        if ((dims[a] - 1) % q != 0 || (dims[a] - 1) / q < 2)
            return fail("every dims[a] must equal c*2^(levels-1)+1 with c >= 2");
    }
    P.ndim = ndim; P.levels = levels; P.esize = int(dt); P.var = (st == HOMG_DIFFUSION7); P.pow2 = pow2;
    P.g.clear(); P.n_alloc.clear();
    size_t es = size_t(dt);
    size_t row_align = 128 / es;           // elements per 128 B
    size_t total = 0;
    for (int m = 0; m < levels; ++m) {
        LevelGeom g;
        int64_t n[3] = {1, 1, 1};
        for (int a = 0; a < ndim; ++a) n[3 - ndim + a] = ((dims[a] - 1) >> m) + 1;
        if (pow2 && m >= 1) n[1] = n[2] = (dims[0] >> m) + 1;            // an anchored lattice of the (N+1)-node grid
        g.nz = int(n[0]); g.ny = int(n[1]); g.nx = int(n[2]);
        g.px = int(round_up(size_t(g.nx), row_align));
        g.pp = (long long)g.px * g.ny;
        size_t na = size_t(g.pp) * size_t(g.nz) + size_t(g.px);        // + one spare row
        na = round_up(na * es, 256) / es;
        P.g.push_back(g);
        P.n_alloc.push_back(na);
        size_t arrays;
        if (pow2 && m >= 1) arrays = 4;                                   // the four anchored source arrays
        else if (m == 0) arrays = 3 /*rot*/ + 3 /*u f g*/ + (P.var ? 5 : 0) /*k fz fy fx wd*/;
        else arrays = kNumRot + 4 /*a g d0 tmp*/ + (P.var ? 5 : 0);
        total += arrays * na * es;
    }
    const LevelGeom& g0 = P.g[0];
    P.staging_bytes = round_up(size_t(g0.nx) * g0.ny * g0.nz * es, 256);
    // one partial per block of the generic residual kernel (32 x 8 x 1 nodes); the fused kernel uses fewer
    P.partial_count = size_t((g0.nx + 31) / 32) * size_t((g0.ny + 7) / 8) * size_t(g0.nz);
    total += P.staging_bytes;
    total += round_up(P.partial_count * sizeof(double), 256);
    total += 256;                           // slot + scalar
    total += 256;                           // front guard
    P.total_bytes = total;                  // + history, added by the caller (depends on options)
    return true;
}

// MFMG schedule: its(m) = min(2^(M-m+1), MaxI), 2 iterations on the coarsest
// level, doubling per finer level.  Visit orders: DESIGN.md R3.
int build_schedule(int kind, int levels, int maxI, const int* xl, const int* xi, int xlen,
                   std::vector<int>& lv, std::vector<int>& it, std::string* why) {
    lv.clear(); it.clear();
    int M = levels - 1;
    auto its = [&](int m) {
        long v = 1L << std::min(M - m + 1, 30);
        return int(std::min<long>(v, maxI));
    };
    if (kind == HOMG_SCHED_EXPLICIT) {
        if (!xl || !xi || xlen < 1) { if (why) *why = "explicit schedule is empty"; return -1; }
        for (int i = 0; i < xlen; ++i) {
            if (xl[i] < 0 || xl[i] > M || xi[i] < 1) { if (why) *why = "explicit schedule entry out of range"; return -1; }
            lv.push_back(xl[i]); it.push_back(xi[i]);
        }
        if (lv.back() != 0) { if (why) *why = "schedule must end on level 0"; return -1; }
        return int(lv.size());
    }
    if (kind == HOMG_SCHED_C) {
        lv.push_back(M);
        for (int k = M - 1; k >= 0; --k) { lv.push_back(k); if (k > 0) lv.push_back(k + 1); }
    } else if (kind == HOMG_SCHED_A) {
        lv.push_back(M);
        if (M >= 1) lv.push_back(M - 1);
        for (int k = M - 2; k >= 0; --k) { lv.push_back(k + 2); lv.push_back(k + 1); lv.push_back(k); }
    } else if (kind == HOMG_SCHED_SAWTOOTH) {
        for (int k = M; k >= 0; --k)
            for (int j = M; j >= k; --j) lv.push_back(j);
    } else {
        if (why) *why = "unknown schedule kind";
        return -1;
    }
    for (size_t i = 0; i < lv.size(); ++i) it.push_back(its(lv[i]));
    return int(lv.size());
}

}  // namespace homg
