// homg_visit3.cuh — K_visit for 3-D levels: one whole MFMG visit (interpolate + correct + NS Jacobi sweeps
// [+ u += e] or [+ S3e bookkeeping]) in ONE pass over HBM.            (Eq. 2-3)
//
// Same pipeline as homg_visit.cuh (which keeps the 2-D form): a CTA owns an x/y tile, marches along z and
// keeps the NS sweeps in flight — at step q the plane z0 = zs+q of v^0 arrives and stage s computes plane
// z0-s of v^s from planes z0-s-1, z0-s, z0-s+1 of v^{s-1}; the tile carries a halo of NS nodes per side that
// is recomputed.  What differs is the work per thread, chosen from the r01 profile (issue-bound at 81
// instructions and 18 shared-memory cycles per warp, pack and stage; profiles/r01e_ncu_full_cfg4.md):
//   * a thread owns TWO adjacent rows of one 16-byte pack (8 fp32 / 4 fp64 nodes per plane): the y neighbours
//     between its two rows are registers, so a stage costs 2 LDS.128 + 2 STS.128 per 2 packs instead of 4 + 2;
//   * g of a plane is read from its TMA ring ONCE into registers and carried down the stages as a register
//     chain (stage s needs g of plane z0-s), instead of one LDS.128 per pack and stage;
//   * the Dirichlet condition is a per-thread multiplier: w_p (Eq. 3) is 0 on boundary / out-of-range nodes,
//     so v stays exactly 0 there (v^0 is 0 there by TMA zero fill) and the steady loop has no selects;
//   * the step loop is unrolled by 4 = the depth of every TMA ring, so ring slots, the parity of z0 (coarse
//     plane pair of the interpolation) and the stage-buffer slot are compile-time constants;
//   * 384 threads (16 packs x 24 row pairs), one CTA per SM at <= 168 registers; tile 64 x 48 nodes (fp32) of
//     which 56 x 40 are stored (NS = 4).
// The arithmetic per node is the expression tree of homg_kernels.cuh (R14): results are bit-identical
// to NS launches of the single-sweep kernels and to the oracle.
#pragma once
#include "homg_fused.cuh"

namespace homg {

// BOOK: the visit of a level >= 1 (S3e bookkeeping, three iterates stored) carries more live values per thread
// (226 registers): 256 threads (16 row pairs, tile 64 x 32) instead of 384 at <= 168.  (320 threads get no more
// registers than 384: ptxas allots them per group of four warps.)
// VAR: the variable-coefficient stencil (flux form, R11) keeps three more TMA rings (the face arrays) and
// more registers per thread: 12 row pairs = 192 threads, tile 16 packs x 24 rows (257^3 fp64: 10 x 13 = 130 tiles)
#ifndef HOMG_VISIT3_VAR_TR
#define HOMG_VISIT3_VAR_TR 12
#endif
template <class T, int NS, bool BOOK, bool VAR = false>
struct Visit3Tile {
    static constexpr int ES = int(sizeof(T));
    static constexpr int VEC = 16 / ES;
    static constexpr int PX = 16, TR = VAR ? HOMG_VISIT3_VAR_TR : (BOOK ? 16 : 24), NT = PX * TR;   // packs per row, row pairs, threads
    static constexpr int HX = (NS + VEC - 1) / VEC * VEC;      // x halo (nodes), pack granular
    static constexpr int HY = (NS + 1) / 2 * 2;                // y halo (rows), row-pair granular
    static constexpr int TXN = PX * VEC, PY = 2 * TR;          // tile in nodes
    static constexpr int OX = TXN - 2 * HX, OY = PY - 2 * HY;  // nodes stored per plane
    static constexpr int RS = TXN;                             // row stride (elements) = 256 B
    static constexpr int ROFF = RS;                            // one pad row below and above the tile
    static constexpr int PLANE = PY * RS + 2 * ROFF;
    static constexpr int PLANE_BYTES = PLANE * ES;
    static constexpr int BOX_BYTES = PY * RS * ES;             // one TMA box {TXN, PY, 1}
    static constexpr int NIN = 4, NG = 4, NC = 4, UNR = 4;     // ring depths = unroll
    // coarse tiles of e_c and a_c (INTERP): the box starts 16-B aligned, hence the slack columns
    static constexpr int CWN = TXN / 2 + 1;
    static constexpr int CW = (CWN + 2 * (VEC - 1)) / VEC * VEC;
    static constexpr int CR = PY / 2 + 1;
    static constexpr int CBOX_BYTES = CR * CW * ES;
    static constexpr int CTILE_BYTES = (CBOX_BYTES + 127) / 128 * 128;
    // epilogue operands (u; or v^0, d0, a) of a step: one 16-byte slot per thread and row, filled by cp.async at the
    // start of the step and read after the NS stages (up to 3 arrays)
    static constexpr int EP_BYTES = 2 * NT * 16;
    static constexpr int NEP = BOOK ? 6 : 0;                   // BOOK: 3 arrays x 2 slots
    // level 0: the stored region of u, one TMA box {OX, OY, 1} per step, NU slots (issued two steps ahead)
    static constexpr int NU = 4;
    static constexpr int UBOX_BYTES = OX * OY * ES;
    static_assert(UBOX_BYTES % 128 == 0 && (OX * ES) % 16 == 0, "u box: 128-B aligned slots, 16-B rows");
    static_assert(CW >= CWN + VEC - 1, "coarse tile too narrow");
    static_assert(PLANE_BYTES % 128 == 0 && BOX_BYTES % 128 == 0, "TMA destinations are 128-B aligned");
    static_assert(NIN == UNR && NG == UNR && NC == UNR, "ring slots are compile-time constants of the unrolled loop");
};

template <class T, int NS, bool INTERP, bool BOOK, bool VAR = false>
__host__ __device__ constexpr int visit3_smem_bytes() {
    using TL = Visit3Tile<T, NS, BOOK, VAR>;
    return TL::NG * TL::BOX_BYTES +
           (INTERP ? TL::NC * 2 * TL::CTILE_BYTES + NS * 2 * TL::PLANE_BYTES
                   : TL::NIN * TL::PLANE_BYTES + (NS - 1) * 2 * TL::PLANE_BYTES) + TL::NEP * TL::EP_BYTES + (BOOK ? 0 : TL::NU * TL::UBOX_BYTES) +
           (VAR ? 4 * TL::NG * TL::BOX_BYTES : 0) + 128;
}

// cp.async (LDGSTS): 16 bytes global -> shared without passing through registers; completion per thread
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }

// ---- one Jacobi stage on a pack: out = v + w_p ((sum_nb v - 2d v) + h^2 g), Eq. 3 in the order of DESIGN.md R14 ----
// generic (fp64): one scalar operation per node and term
template <class T>
__device__ __forceinline__ Pack<T> jacobi_pack(const Pack<T>& pv, const Pack<T>& cu, const Pack<T>& nx, const Pack<T>& dn,
                                               const Pack<T>& up, const Pack<T>& gv, T vl, T vr, const Pack<T>& wpm,
                                               const Coef<T>& cf) {
    constexpr int VEC = 16 / int(sizeof(T));
    Pack<T> out;
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
        const T vc = cu.v[j];
        const T xm = j == 0 ? vl : cu.v[j - 1 < 0 ? 0 : j - 1];
        const T xp = j == VEC - 1 ? vr : cu.v[j + 1 > VEC - 1 ? VEC - 1 : j + 1];
        T sm = pv.v[j] + nx.v[j];
        sm += dn.v[j] + up.v[j];
        sm += xm + xp;
        T t = fma_rn(-cf.twod, vc, sm);
        t = fma_rn(cf.h2, gv.v[j], t);
        out.v[j] = fma_rn(wpm.v[j], t, vc);
    }
    return out;
}
// fp32: sm_100a packed pairs (add / fma .rn.f32x2 = FADD2 / FFMA2: two IEEE round-to-nearest operations per
// instruction, so the results are those of the scalar form bit for bit).  A pack is two pairs (v0,v1), (v2,v3) —
// the register pairs LDS.128 / STS.128 already use; only the x-neighbour sums (vl+v1, v0+v2), (v1+v3, v2+vr) pair
// nodes differently and are formed by four scalar additions.  18 instructions per pack instead of 32.
__device__ __forceinline__ Pack<float> jacobi_pack(const Pack<float>& pv, const Pack<float>& cu, const Pack<float>& nx,
                                                   const Pack<float>& dn, const Pack<float>& up, const Pack<float>& gv,
                                                   float vl, float vr, const Pack<float>& wpm, const Coef<float>& cf) {
    const F2 ntd = f2_make(-cf.twod, -cf.twod), h2 = f2_make(cf.h2, cf.h2);
    const float xs[4] = {vl + cu.v[1], cu.v[0] + cu.v[2], cu.v[1] + cu.v[3], cu.v[2] + vr};
    Pack<float> out;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const F2 c2 = f2_make(cu.v[2 * h], cu.v[2 * h + 1]);
        F2 sm = f2_add(f2_make(pv.v[2 * h], pv.v[2 * h + 1]), f2_make(nx.v[2 * h], nx.v[2 * h + 1]));
        sm = f2_add(sm, f2_add(f2_make(dn.v[2 * h], dn.v[2 * h + 1]), f2_make(up.v[2 * h], up.v[2 * h + 1])));
        sm = f2_add(sm, f2_make(xs[2 * h], xs[2 * h + 1]));
        F2 t = f2_fma(ntd, c2, sm);
        t = f2_fma(h2, f2_make(gv.v[2 * h], gv.v[2 * h + 1]), t);
        f2_get(f2_fma(f2_make(wpm.v[2 * h], wpm.v[2 * h + 1]), t, c2), out.v[2 * h], out.v[2 * h + 1]);
    }
    return out;
}

// variable coefficient (flux form, R11/R14): v + (g - A v) wd with A v = sum_faces kf (v - v_nb) / h^2 (faces in the order
// z-, z+, y-, y+, x-, x+: A v is the very number k_relax_tma<VAR> / the oracle compute) and wd = RN(w / D) precomputed per
// node in S0 (k_wdiag).  The per-sweep kernels and the oracle evaluate v + w (g - A v) / D: the two differ by rounding only
// (one multiplication by a rounded quotient instead of a multiplication and a division) — DESIGN.md R14, tolerance 1e-12.
// Without the sum of the faces and the IEEE division the dependent chain per node is 2.7 x shorter: with 6 warps per SM the
// kernel is bound by exactly that latency (profiles/r02b).  fxl = the x- face of the pack's first node.
template <class T>
__device__ __forceinline__ Pack<T> jacobi_pack_var(const Pack<T>& pv, const Pack<T>& cu, const Pack<T>& nx, const Pack<T>& dn,
                                                   const Pack<T>& up, const Pack<T>& gv, T vl, T vr, const Pack<T>& wd,
                                                   const Pack<T>& fzm, const Pack<T>& fzp, const Pack<T>& fym, const Pack<T>& fyp,
                                                   const Pack<T>& fxp, T fxl, const Coef<T>& cf) {
    constexpr int VEC = 16 / int(sizeof(T));
    Pack<T> out;
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
        const T vc = cu.v[j];
        const T xm = j == 0 ? vl : cu.v[j - 1 < 0 ? 0 : j - 1];
        const T xp = j == VEC - 1 ? vr : cu.v[j + 1 > VEC - 1 ? VEC - 1 : j + 1];
        const T fxm = j == 0 ? fxl : fxp.v[j - 1 < 0 ? 0 : j - 1];
        T acc = T(0);
        acc += fzm.v[j] * (vc - pv.v[j]);
        acc += fzp.v[j] * (vc - nx.v[j]);
        acc += fym.v[j] * (vc - dn.v[j]);
        acc += fyp.v[j] * (vc - up.v[j]);
        acc += fxm * (vc - xm);
        acc += fxp.v[j] * (vc - xp);
        const T Av = acc * cf.ih2;
        out.v[j] = vc + (gv.v[j] - Av) * wd.v[j];                  // wd = 0 on the boundary and outside the grid: v stays 0
    }
    return out;
}

// q mod UNR of a step: a compile-time constant in the steady loop, q itself elsewhere
template <int N>
__device__ __forceinline__ constexpr int step_k(std::integral_constant<int, N>) { return N; }
__device__ __forceinline__ int step_k(int q) { return q; }

// Arguments as k_visit (homg_visit.cuh).  grid = (x tiles of OX, y tiles of OY, z chunks of mchunk interior
// planes); mchunk must be even when there is more than one chunk (every chunk then starts on an odd plane).
// VAR: tm_fz / tm_fy / tm_fx = the face arrays of the level (box {TXN, PY, 1} like g); otherwise unused.
template <class T, int NS, bool INTERP, bool BOOK, bool VAR = false>
__global__ void __launch_bounds__(Visit3Tile<T, NS, BOOK, VAR>::NT, 1)
k_visit3(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_ac,
         const __grid_constant__ CUtensorMap tm_g, const __grid_constant__ CUtensorMap tm_u,
         const __grid_constant__ CUtensorMap tm_fz, const __grid_constant__ CUtensorMap tm_fy,
         const __grid_constant__ CUtensorMap tm_fx, const __grid_constant__ CUtensorMap tm_wd, LevelGeom g, Coef<T> cf,
         T* __restrict__ o0,
         T* __restrict__ o1, T* __restrict__ o2, T* __restrict__ a, int a_assign, const T* __restrict__ d0,
         const T* __restrict__ v0, T* __restrict__ u, int mchunk) {
    pdl_start();
    static_assert(!(INTERP && BOOK), "interpolate+correct is fused on level 0 only");
    static_assert(!(VAR && BOOK), "the variable-coefficient form runs level-0 visits only");
    using TL = Visit3Tile<T, NS, BOOK, VAR>;
    constexpr int VEC = TL::VEC, RS = TL::RS;
    const int tid = threadIdx.x, px = tid % TL::PX, tr = tid / TL::PX;
    const int NM = g.nz;
    const long long mstride = g.pp;
    const int x0 = blockIdx.x * TL::OX, y0 = blockIdx.y * TL::OY;
    const int ms = 1 + blockIdx.z * mchunk;
    const int me = min(ms + mchunk, NM - 1);
    if (ms >= me) return;
    const int zs = ms - NS;                                        // first plane of stage 0 (ms is odd)
    const int nsteps = me - ms + 2 * NS;                           // one stage-0 plane per step
    const int Zc0 = zs >> 1;                                       // first coarse plane (floor)
    const int ncz = ((me + NS) >> 1) - Zc0 + 1;

    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    __shared__ uint64_t fbar[TL::NIN], gbar[TL::NG], cbar[TL::NC], ubar[TL::NU], sbar;
    auto gs = [&](int st) { return reinterpret_cast<T*>(smem + st * TL::BOX_BYTES); };
    unsigned char* cbase = smem + TL::NG * TL::BOX_BYTES;          // PLAIN: v ring;  INTERP: coarse ring
    auto vring = [&](int st) { return reinterpret_cast<T*>(cbase + st * TL::PLANE_BYTES); };
    auto ce = [&](int st) { return reinterpret_cast<T*>(cbase + (2 * st) * TL::CTILE_BYTES); };
    auto ca = [&](int st) { return reinterpret_cast<T*>(cbase + (2 * st + 1) * TL::CTILE_BYTES); };
    unsigned char* sbase = cbase + (INTERP ? TL::NC * 2 * TL::CTILE_BYTES : TL::NIN * TL::PLANE_BYTES);
    constexpr int NBUF = INTERP ? NS : NS - 1;
    unsigned char* epbase = sbase + NBUF * 2 * TL::PLANE_BYTES;
    auto eps = [&](int arr, int r) { return reinterpret_cast<T*>(epbase + arr * TL::EP_BYTES + (r * TL::NT + tid) * 16); };
    auto us = [&](int st) { return reinterpret_cast<T*>(epbase + TL::NEP * TL::EP_BYTES + st * TL::UBOX_BYTES); };
    const bool stage_u = !BOOK && u != nullptr;
    // VAR: rings of the face planes, slot = that of g (order fz, fy, fx: fy is read one row below, fx one element left)
    unsigned char* fcbase = epbase + TL::NEP * TL::EP_BYTES + (BOOK ? 0 : TL::NU * TL::UBOX_BYTES);
    auto fcs = [&](int arr, int st) { return reinterpret_cast<T*>(fcbase + (arr * TL::NG + st) * TL::BOX_BYTES); };
    auto buf = [&](int s, int slot) {                              // plane published by stage s
        return reinterpret_cast<T*>(sbase + ((INTERP ? s : s - 1) * 2 + slot) * TL::PLANE_BYTES);
    };

    if (tid == 0) {
        for (int s = 0; s < TL::NIN; ++s) mbar_init(&fbar[s], 1);
        for (int s = 0; s < TL::NG; ++s) mbar_init(&gbar[s], 1);
        for (int s = 0; s < TL::NC; ++s) mbar_init(&cbar[s], 1);
        mbar_init(&sbar, TL::NT);
        for (int s = 0; s < TL::NU; ++s) mbar_init(&ubar[s], 1);
        mbar_fence_init();
    }
    // the pad rows of every plane are read as the y neighbours of the first / last tile row (halo rows whose
    // results are never used): keep them finite
    {
        constexpr int NPL = (INTERP ? 0 : TL::NIN) + NBUF * 2;
        unsigned char* pl0 = INTERP ? sbase : cbase;
        for (int i = tid; i < NPL * 2 * TL::ROFF; i += TL::NT) {
            const int p = i / (2 * TL::ROFF), r = i - p * 2 * TL::ROFF;
            T* pl = reinterpret_cast<T*>(pl0 + p * TL::PLANE_BYTES);
            pl[r < TL::ROFF ? r : TL::ROFF + TL::PY * RS + (r - TL::ROFF)] = T(0);
        }
    }
    __syncthreads();

    const int Xc = (x0 - TL::HX) / 2;                              // x0 - HX is even
    const int Xa = Xc - (Xc & (VEC - 1));                          // coarse box start, 16-B aligned
    const int Yc = (y0 - TL::HY) >> 1;                             // y0 - HY is even
    auto issue_v = [&](int i) {                                    // PLAIN: plane zs+i of v^0
        const int st = i & (TL::NIN - 1);
        mbar_arrive_expect_tx(&fbar[st], TL::BOX_BYTES);
        tma_load_3d(vring(st) + TL::ROFF, &tm_in, &fbar[st], x0 - TL::HX, y0 - TL::HY, zs + i);
    };
    auto issue_g = [&](int i) {                                    // plane zs+i of g (read at step i+1)
        const int st = i & (TL::NG - 1);
        mbar_arrive_expect_tx(&gbar[st], (VAR ? 5 : 1) * TL::BOX_BYTES);
        tma_load_3d(gs(st), &tm_g, &gbar[st], x0 - TL::HX, y0 - TL::HY, zs + i);
        if (VAR) {
            tma_load_3d(fcs(0, st), &tm_fz, &gbar[st], x0 - TL::HX, y0 - TL::HY, zs + i);
            tma_load_3d(fcs(1, st), &tm_fy, &gbar[st], x0 - TL::HX, y0 - TL::HY, zs + i);
            tma_load_3d(fcs(2, st), &tm_fx, &gbar[st], x0 - TL::HX, y0 - TL::HY, zs + i);
            tma_load_3d(fcs(3, st), &tm_wd, &gbar[st], x0 - TL::HX, y0 - TL::HY, zs + i);
        }
    };
    auto issue_u = [&](int i) {                                    // stored region of u at the plane step i finishes
        const int st = i & (TL::NU - 1);
        mbar_arrive_expect_tx(&ubar[st], TL::UBOX_BYTES);
        tma_load_3d(us(st), &tm_u, &ubar[st], x0, y0, zs + i - NS);
    };
    auto issue_c = [&](int zc) {                                   // coarse plane Zc0+zc of e_c and a_c
        const int st = zc & (TL::NC - 1);
        mbar_arrive_expect_tx(&cbar[st], 2 * TL::CBOX_BYTES);
        tma_load_3d(ce(st), &tm_in, &cbar[st], Xa, Yc, Zc0 + zc);
        tma_load_3d(ca(st), &tm_ac, &cbar[st], Xa, Yc, Zc0 + zc);
    };
    if (tid == 0) {
        if (INTERP)
            for (int zc = 0; zc < TL::NC && zc < ncz; ++zc) issue_c(zc);
        for (int i = 0; i < TL::NIN - 1 && i < nsteps; ++i) {
            if (!INTERP) issue_v(i);
            if (i <= nsteps - 2) issue_g(i);
            if (stage_u) issue_u(i);
        }
    }

    // ---- this thread: pack x .. x+VEC-1 of rows ye (even tile row 2 tr) and ye+1 ----
    const int x = x0 - TL::HX + px * VEC;
    const int ye = y0 - TL::HY + 2 * tr;
    const int offE = TL::ROFF + (2 * tr) * RS + px * VEC, offO = offE + RS;   // in a padded plane
    const int goffE = (2 * tr) * RS + px * VEC, goffO = goffE + RS;
    // Eq. 3 multiplier w_p of every node; 0 where the node is not an interior node of the level
    Pack<T> wpm[2];
    bool own[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int y = ye + r;
        const bool row_int = y > 0 && y < g.ny - 1;
#pragma unroll
        for (int j = 0; j < VEC; ++j) wpm[r].v[j] = (row_int && x + j > 0 && x + j < g.nx - 1) ? cf.wp : T(0);
        own[r] = px * VEC >= TL::HX && px * VEC < TL::HX + TL::OX && x < g.nx && 2 * tr + r >= TL::HY &&
                 2 * tr + r < TL::HY + TL::OY && y < g.ny;
    }
    const int uoff = (2 * tr - TL::HY) * TL::OX + px * VEC - TL::HX;   // my even row in a u box (own threads only)
    const int coff = tr * TL::CW + (Xc - Xa) + px * (VEC / 2);     // INTERP: my first coarse node, coarse row ye/2

    // S3a in registers: the two packs of v^0 at fine plane z (rows ye even, ye+1 odd) from the coarse planes
    // z>>1 and (z+1)>>1; summation order as homg_first.cuh / the oracle: rows (z lo, y lo), (z lo, y hi),
    // (z hi, y lo), (z hi, y hi)
    auto produce = [&](const int z, const bool zodd, Pack<T>* out) {
        constexpr int NCV = VEC / 2 + 1;
        const int zlo = (z >> 1) - Zc0, zhi = ((z + 1) >> 1) - Zc0;
        mbar_wait(&cbar[zlo & (TL::NC - 1)], (zlo / TL::NC) & 1);
        if (zodd) mbar_wait(&cbar[zhi & (TL::NC - 1)], (zhi / TL::NC) & 1);
        const T* A0 = ca(zlo & (TL::NC - 1)) + coff;
        const T* A1 = ca(zhi & (TL::NC - 1)) + coff;
        const T* E0 = ce(zlo & (TL::NC - 1)) + coff;
        auto ldrow = [&](const T* rp, T* c) {
            if (VEC == 4) {
                const HalfPack<T> h = *reinterpret_cast<const HalfPack<T>*>(rp);
                c[0] = h.v[0]; c[1] = h.v[1]; c[NCV - 1] = rp[NCV - 1];
            } else {
#pragma unroll
                for (int i = 0; i < NCV; ++i) c[i] = rp[i];
            }
        };
        auto addrow = [&](T* acc, const T* c, const bool first) {
#pragma unroll
            for (int j = 0; j < VEC; ++j) {
                if (j & 1) { acc[j] = first ? c[j >> 1] : acc[j] + c[j >> 1]; acc[j] += c[(j >> 1) + 1]; }
                else acc[j] = first ? c[j >> 1] : acc[j] + c[j >> 1];
            }
        };
        T c00[NCV], c01[NCV], c10[NCV], c11[NCV], accE[VEC], accO[VEC];
        ldrow(A0, c00);
        ldrow(A0 + TL::CW, c01);
        if (zodd) { ldrow(A1, c10); ldrow(A1 + TL::CW, c11); }
        addrow(accE, c00, true);
        addrow(accO, c00, true);
        addrow(accO, c01, false);
        if (zodd) {
            addrow(accE, c10, false);
            addrow(accO, c10, false);
            addrow(accO, c11, false);
        }
        const T wE = zodd ? T(0.5) : T(1), wO = zodd ? T(0.25) : T(0.5);
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
            if (j & 1) { out[0].v[j] = (T(0.5) * wE) * accE[j]; out[1].v[j] = (T(0.5) * wO) * accO[j]; }
            else { out[0].v[j] = zodd ? wE * accE[j] : E0[j >> 1]; out[1].v[j] = wO * accO[j]; }
        }
    };

    // register state: own columns of every stage input (previous and current plane), g of the stages
    Pack<T> P[NS][2], C[NS][2], Gh[NS - 1][2];
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
#pragma unroll
            for (int s = 0; s < NS; ++s) { P[s][r].v[j] = T(0); C[s][r].v[j] = T(0); }
#pragma unroll
            for (int s = 0; s < NS - 1; ++s) Gh[s][r].v[j] = T(0);
        }

    // VAR: faces of the plane stage s works on, carried from stage to stage like g (stage s reads the plane stage s-1
    // read one step earlier): z+ faces of my two rows, y faces of rows ye-1, ye, ye+1, x+ faces of my two rows and
    // the x- face of each pack's first node; and the z- face of every stage = the z+ face it used one step ago
    constexpr int NF = VAR ? NS - 1 : 1, NZ = VAR ? NS : 1;
    Pack<T> Fzh[NF][2], Fyh[NF][3], Fxh[NF][2], Fzm[NZ][2], Wdh[NF][2];
    T Fxlh[NF][2];
    if (VAR) {
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
#pragma unroll
            for (int s = 0; s < NF; ++s) {
                Fzh[s][0].v[j] = Fzh[s][1].v[j] = Fxh[s][0].v[j] = Fxh[s][1].v[j] = Wdh[s][0].v[j] = Wdh[s][1].v[j] = T(0);
                Fyh[s][0].v[j] = Fyh[s][1].v[j] = Fyh[s][2].v[j] = T(0);
                Fxlh[s][0] = Fxlh[s][1] = T(0);
            }
#pragma unroll
            for (int s = 0; s < NZ; ++s) Fzm[s][0].v[j] = Fzm[s][1].v[j] = T(0);
        }
    }

    // address of (x, ye) in the plane the LAST stage produces at step q: z = zs + q - NS
    long long cF = (long long)(zs - NS) * mstride + (long long)ye * g.px + x;
    const long long rowO = g.px;

    // One step.  kq: q mod UNR as an integral_constant (STEADY: every slot below folds to a constant) or q itself.
    auto step = [&](auto kq, auto SD, const int q) {
        constexpr bool STEADY = decltype(SD)::value;
        const int K = step_k(kq);
        const int W = K & 1, R = W ^ 1;                            // stage-buffer slots: written now / read now
        const int KV = K & (TL::NIN - 1), KP = (K + TL::NIN - 1) & (TL::NIN - 1);   // ring slots of planes q, q-1
        const int z0 = zs + q;
        const bool zodd = (1 + NS + K) & 1;                        // parity of z0 (ms is odd)
        // ---- stage 0: the packs of v^0 at plane z0 (registers only, so far) ----
        Pack<T> nx[2];
        if (INTERP) {
            produce(z0, zodd, nx);
        } else {
            mbar_wait(&fbar[KV], (q / TL::NIN) & 1);
            nx[0] = *reinterpret_cast<const Pack<T>*>(vring(KV) + offE);
            nx[1] = *reinterpret_cast<const Pack<T>*>(vring(KV) + offO);
        }
        // ---- every thread has finished the shared-memory traffic of step q-1 (it arrived after its last stage
        // store; its last stage, its epilogue and the stage 0 above hide the skew between warps) ----
        if (STEADY || q >= 1) {
            mbar_wait(&sbar, R);
            if (tid == 0) {                                        // ring slots of planes q-1 are free: refill
                const int i = q + TL::NIN - 2;
                if (!INTERP && i < nsteps) issue_v(i);
                if (i <= nsteps - 2) issue_g(i);
                if (stage_u && q + 2 < nsteps) issue_u(q + 2);     // (its slot was last read in step q-2)
                if (INTERP && !zodd) {                             // plane z0-1 was odd: coarse plane (z0-1)>>1 is dead
                    const int zc = ((z0 - 1) >> 1) - Zc0 + TL::NC;
                    if (zc < ncz) issue_c(zc);
                }
            }
        }
        if (INTERP) {
            *reinterpret_cast<Pack<T>*>(buf(0, W) + offE) = nx[0];
            *reinterpret_cast<Pack<T>*>(buf(0, W) + offO) = nx[1];
        }
        const bool fin = STEADY || q >= 2 * NS;
        // operands of the NEXT step's epilogue (u; or v^0, d0, a): global -> shared by cp.async, one step ahead into
        // the other slot (no registers; with ~200 KB of shared memory there is no L1 left to prefetch into).
        // One group per step.
        {
            const bool pre = STEADY || (q + 1 >= 2 * NS && q + 1 < nsteps);
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                if (!own[r] || !pre) continue;
                const long long c = cF + r * rowO + mstride;
                if (BOOK && a) {
                    cp_async16(eps(R, r), v0 + c);
                    if (d0) cp_async16(eps(2 + R, r), d0 + c);
                    if (!a_assign) cp_async16(eps(4 + R, r), a + c);
                }
            }
            if (BOOK) cp_async_commit();
        }
        // g of plane z0-1: from its ring into registers, once; stage s reads it s-1 steps from now
        Pack<T> gn[2];
        if (STEADY || q >= 1) {
            mbar_wait(&gbar[KP], ((q - 1) / TL::NG) & 1);
            gn[0] = *reinterpret_cast<const Pack<T>*>(gs(KP) + goffE);
            gn[1] = *reinterpret_cast<const Pack<T>*>(gs(KP) + goffO);
        } else {
#pragma unroll
            for (int j = 0; j < VEC; ++j) { gn[0].v[j] = T(0); gn[1].v[j] = T(0); }
        }
        // VAR: the faces of plane z0-1 (same ring slot, same barrier as g)
        Pack<T> fzn[2], fyn[3], fxn[2], wdn[2];
        T fxln[2] = {T(0), T(0)};
        if (VAR) {
            if (STEADY || q >= 1) {
                fzn[0] = *reinterpret_cast<const Pack<T>*>(fcs(0, KP) + goffE);
                fzn[1] = *reinterpret_cast<const Pack<T>*>(fcs(0, KP) + goffO);
                fyn[0] = *reinterpret_cast<const Pack<T>*>(fcs(1, KP) + goffE - RS);
                fyn[1] = *reinterpret_cast<const Pack<T>*>(fcs(1, KP) + goffE);
                fyn[2] = *reinterpret_cast<const Pack<T>*>(fcs(1, KP) + goffO);
                fxn[0] = *reinterpret_cast<const Pack<T>*>(fcs(2, KP) + goffE);
                fxn[1] = *reinterpret_cast<const Pack<T>*>(fcs(2, KP) + goffO);
                wdn[0] = *reinterpret_cast<const Pack<T>*>(fcs(3, KP) + goffE);
                wdn[1] = *reinterpret_cast<const Pack<T>*>(fcs(3, KP) + goffO);
                fxln[0] = fcs(2, KP)[goffE - 1];
                fxln[1] = fcs(2, KP)[goffO - 1];
            } else {
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    fzn[0].v[j] = fzn[1].v[j] = fxn[0].v[j] = fxn[1].v[j] = wdn[0].v[j] = wdn[1].v[j] = T(0);
                    fyn[0].v[j] = fyn[1].v[j] = fyn[2].v[j] = T(0);
                }
            }
        }
        // y neighbours across threads: row ye-1 (below my even row) and row ye+2 (above my odd row), published in
        // the previous step.  Those of stage s+1 are fetched BEFORE stage s stores (the compiler cannot move a
        // shared load above a shared store by itself).
        auto fetch = [&](const int s, Pack<T>& dn, Pack<T>& up) {
            const T* ctr = (s == 1 && !INTERP) ? vring(KP) : buf(s - 1, R);
            dn = *reinterpret_cast<const Pack<T>*>(ctr + offE - RS);
            up = *reinterpret_cast<const Pack<T>*>(ctr + offO + RS);
        };
        constexpr bool AHEAD = !BOOK;                              // (the bookkeeping form has no registers to spare)
        Pack<T> dnN, upN;
        if (AHEAD) fetch(1, dnN, upN);
#pragma unroll
        for (int s = 1; s <= NS; ++s) {
            // stage s: plane z0-s of v^s from v^{s-1}: P (z0-s-1), C (z0-s), nx (z0-s+1)
            if (!AHEAD) fetch(s, dnN, upN);
            const Pack<T> dnE = dnN, upO = upN;
            if (AHEAD && s < NS) fetch(s + 1, dnN, upN);
            const int z = z0 - s;
            const bool zin = STEADY || (z > 0 && z < NM - 1);
            Pack<T> out[2];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const Pack<T> cu = C[s - 1][r], pv = P[s - 1][r];
                const Pack<T>& dn = r == 0 ? dnE : C[s - 1][0];
                const Pack<T>& up = r == 0 ? C[s - 1][1] : upO;
                const Pack<T>& gv = s == 1 ? gn[r] : Gh[s == 1 ? 0 : s - 2][r];
                const T vl = __shfl_up_sync(0xffffffffu, cu.v[VEC - 1], 1);
                const T vr = __shfl_down_sync(0xffffffffu, cu.v[0], 1);
                if (VAR) {
                    const Pack<T>& fzp = s == 1 ? fzn[r] : Fzh[s == 1 ? 0 : s - 2][r];
                    const Pack<T>& fym = s == 1 ? fyn[r] : Fyh[s == 1 ? 0 : s - 2][r];
                    const Pack<T>& fyp = s == 1 ? fyn[r + 1] : Fyh[s == 1 ? 0 : s - 2][r + 1];
                    const Pack<T>& fxp = s == 1 ? fxn[r] : Fxh[s == 1 ? 0 : s - 2][r];
                    const T fxl = s == 1 ? fxln[r] : Fxlh[s == 1 ? 0 : s - 2][r];
                    const Pack<T>& wdv = s == 1 ? wdn[r] : Wdh[s == 1 ? 0 : s - 2][r];
                    out[r] = jacobi_pack_var(pv, cu, nx[r], dn, up, gv, vl, vr, wdv, Fzm[s - 1][r], fzp, fym, fyp, fxp, fxl, cf);
                    Fzm[s - 1][r] = fzp;                          // the z- face of this stage's next plane
                } else {
                    out[r] = jacobi_pack(pv, cu, nx[r], dn, up, gv, vl, vr, wpm[r], cf);
                }
                if (!zin) {                                        // Dirichlet planes z = 0, nz-1 (and beyond)
#pragma unroll
                    for (int j = 0; j < VEC; ++j) out[r].v[j] = T(0);
                }
            }
            if (s < NS) {
                *reinterpret_cast<Pack<T>*>(buf(s, W) + offE) = out[0];
                *reinterpret_cast<Pack<T>*>(buf(s, W) + offO) = out[1];
            }
            // all shared-memory traffic of this step that other threads see is done (stage NS's neighbours were
            // fetched above): arrive now, wait at the end of the step — the last stage and the epilogue hide the skew
            if (s == NS - 1) mbar_arrive(&sbar);
            if (s == NS) {                                         // (every issued u box is waited for: none in flight at exit)
                if (BOOK && fin) cp_async_wait_1();
                if (!BOOK && stage_u) mbar_wait(&ubar[K & (TL::NU - 1)], (q / TL::NU) & 1);
            }
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                if (!own[r]) continue;
                const long long c = cF + r * rowO;
                if (BOOK && s == NS - 2 && s >= 1 && o2 != nullptr && (STEADY || (q >= 2 * NS - 2 && q <= nsteps - 3)))
                    *reinterpret_cast<Pack<T>*>(o2 + c + 2 * mstride) = out[r];
                if (BOOK && s == NS - 1 && s >= 1 && o1 != nullptr && (STEADY || (q >= 2 * NS - 1 && q <= nsteps - 2)))
                    *reinterpret_cast<Pack<T>*>(o1 + c + mstride) = out[r];
                if (s == NS && fin) {
                    if (o0) *reinterpret_cast<Pack<T>*>(o0 + c) = out[r];
                    if (BOOK && a) {                               // S3e: a (+)= d0 + v^{NS-1} - v^0
                        Pack<T> dd, vv = *reinterpret_cast<const Pack<T>*>(eps(W, r)), aa;
                        if (d0) dd = *reinterpret_cast<const Pack<T>*>(eps(2 + W, r));
                        if (!a_assign) aa = *reinterpret_cast<const Pack<T>*>(eps(4 + W, r));
#pragma unroll
                        for (int j = 0; j < VEC; ++j) {
                            const T Dq = ((d0 ? dd.v[j] : T(0)) + C[s - 1][r].v[j]) - vv.v[j];
                            aa.v[j] = a_assign ? Dq : aa.v[j] + Dq;
                        }
                        *reinterpret_cast<Pack<T>*>(a + c) = aa;
                    }
                    if (!BOOK && u) {                              // S4: u += v^NS
                        Pack<T> uu = *reinterpret_cast<const Pack<T>*>(us(K & (TL::NU - 1)) + uoff + r * TL::OX);
#pragma unroll
                        for (int j = 0; j < VEC; ++j) uu.v[j] += out[r].v[j];
                        *reinterpret_cast<Pack<T>*>(u + c) = uu;
                    }
                }
            }
#pragma unroll
            for (int r = 0; r < 2; ++r) { P[s - 1][r] = C[s - 1][r]; C[s - 1][r] = nx[r]; nx[r] = out[r]; }
        }
#pragma unroll
        for (int s = NS - 2; s >= 1; --s) { Gh[s][0] = Gh[s - 1][0]; Gh[s][1] = Gh[s - 1][1]; }
        Gh[0][0] = gn[0]; Gh[0][1] = gn[1];
        if (VAR) {
#pragma unroll
            for (int s = NS - 2; s >= 1; --s) {
                Fzh[s][0] = Fzh[s - 1][0]; Fzh[s][1] = Fzh[s - 1][1]; Fxh[s][0] = Fxh[s - 1][0]; Fxh[s][1] = Fxh[s - 1][1];
                Fyh[s][0] = Fyh[s - 1][0]; Fyh[s][1] = Fyh[s - 1][1]; Fyh[s][2] = Fyh[s - 1][2];
                Fxlh[s][0] = Fxlh[s - 1][0]; Fxlh[s][1] = Fxlh[s - 1][1];
                Wdh[s][0] = Wdh[s - 1][0]; Wdh[s][1] = Wdh[s - 1][1];
            }
            Fzh[0][0] = fzn[0]; Fzh[0][1] = fzn[1]; Fxh[0][0] = fxn[0]; Fxh[0][1] = fxn[1];
            Fyh[0][0] = fyn[0]; Fyh[0][1] = fyn[1]; Fyh[0][2] = fyn[2];
            Fxlh[0][0] = fxln[0]; Fxlh[0][1] = fxln[1];
            Wdh[0][0] = wdn[0]; Wdh[0][1] = wdn[1];
        }
        cF += mstride;
    };
    int q = 0;
    while (q < nsteps) {
        // UNR steps from a multiple of UNR are steady when all their stores are due and every stage's plane is interior
        const bool steady = (q & (TL::UNR - 1)) == 0 && q >= 2 * NS && q + TL::UNR - 1 <= nsteps - 3 &&
                            zs + q - NS >= 1 && zs + q + TL::UNR - 1 <= NM - 2;
        if (steady) {
            step(std::integral_constant<int, 0>{}, std::true_type{}, q);
            step(std::integral_constant<int, 1>{}, std::true_type{}, q + 1);
            step(std::integral_constant<int, 2>{}, std::true_type{}, q + 2);
            step(std::integral_constant<int, 3>{}, std::true_type{}, q + 3);
            q += TL::UNR;
        } else {
            step(q, std::false_type{}, q);
            ++q;
        }
    }
}

}  // namespace homg
