// homg_visit.cuh — K_visit: one whole MFMG visit of a large 3-D level in ONE pass over HBM
// (north_star item 2, taken one step further: interpolate + correct + NS Jacobi sweeps [+ u += e]).
//
// A visit is NS damped-Jacobi sweeps v^s = v^{s-1} + w D^-1 (g - A v^{s-1}), s = 1..NS (PAPER.md
// L53-67, Eq. 2-3), on the same level.  Run as NS launches it moves 3 arrays per sweep.  Here a CTA
// owns an x/y tile, marches along z and keeps a software pipeline of the NS sweeps in flight:
// at step q the plane z0 = zs+q of v^0 arrives, and stage s computes plane z0-s of v^s from the
// planes z0-s-1, z0-s, z0-s+1 of v^{s-1}.  Every thread owns one 16-byte pack of x nodes of one row
// and carries its own column of every v^{s-1} (previous / current / next plane) in registers; the
// in-plane neighbours come from shared memory (y) and warp shuffles (x).  Each stage publishes the
// plane it produced in a 2-slot shared-memory buffer for the next stage's y neighbours, so one
// __syncthreads per step suffices.  The tile carries a halo of NS nodes per side that is
// recomputed (valid region shrinks by one node per stage); only the inner OX x OY nodes are stored.
//
// HBM traffic of a level-0 visit (NS = 4): read g, read the two coarse arrays (INTERP) or v^0,
// read+write u  =  (3 + 2/8) passes instead of (2 + 2/8) + 3 + 3 + 4.
//
// Stage 0 is either PLAIN (v^0 planes staged by TMA) or INTERP (S3a: v^0 built in shared memory
// from the coarse planes of e_c and a_c, as in homg_first.cuh).  Epilogues of the last stage are
// those of k_relax: S3e bookkeeping (a += d0 + v^{NS-1} - v^0) and S4 (u += v^NS); the last three
// iterates can be stored (o0 = v^NS, o1 = v^{NS-1}, o2 = v^{NS-2}) because the next visit's carried
// variation needs them (S3c).
//
// The arithmetic per node is the expression tree of homg_kernels.cuh (R14): results are
// bit-identical to NS launches of the single-sweep kernels and to the oracle.
#pragma once
#include "homg_fused.cuh"

namespace homg {

template <class T, int ND, int NS>
struct VisitTile {
    static constexpr int ES = int(sizeof(T));
    static constexpr int VEC = 16 / ES;
    // 3-D: 16 packs x 32 rows per plane.  2-D: the marching axis is y, a "plane" is one row segment of
    // 160 packs (a width that is NOT close to a power of two: 2^k+1 grids then tile with little waste).
    static constexpr int PX = ND == 3 ? 16 : 160, PY = ND == 3 ? 32 : 1, NT = PX * PY;
    static constexpr int CTAS = ND == 3 ? 1 : 2;              // CTAs per SM (launch bound)
    static constexpr int HX = (NS + VEC - 1) / VEC * VEC;     // x halo (nodes), pack granular
    static constexpr int HY = ND == 3 ? NS : 0;
    static constexpr int TXN = PX * VEC;                      // tile width in nodes
    static constexpr int OX = TXN - 2 * HX, OY = PY - 2 * HY; // nodes stored per plane
    static constexpr int RS = TXN;                            // row stride (elements), a multiple of 128 B
    // padded plane: 3-D one pad row below and above; 2-D 128 B before and after the row
    static constexpr int ROFF = ND == 3 ? RS : 128 / ES;      // where the tile starts inside a padded plane
    static constexpr int PLANE = PY * RS + 2 * ROFF;
    static constexpr int PLANE_BYTES = PLANE * ES;
    static constexpr int BOX_BYTES = PY * RS * ES;            // bytes of one fine plane of the tile
    static constexpr int BW = ND == 3 ? TXN : 160;            // TMA box width (<= 256 elements); TXN / BW boxes per plane
    static constexpr int NIN = 4;                             // TMA ring depth of the v^0 planes
    static constexpr int NGR = 8;                             // g ring: plane z0-s is read by stage s (NS <= 4)
    // coarse tiles of e_c and a_c (INTERP)
    static constexpr int CWN = TXN / 2 + 1;                   // coarse columns a tile row needs
    // + slack: the box starts 16-B aligned.  2-D: three boxes of 512 B
    static constexpr int CBW = ND == 3 ? (CWN + 2 * (VEC - 1)) / VEC * VEC : 512 / ES;
    static constexpr int NCB = ND == 3 ? 1 : 3;
    static constexpr int CW = CBW * NCB;
    static constexpr int CR = ND == 3 ? PY / 2 + 2 : 1;
    static constexpr int CBOX_BYTES = CR * CW * ES;
    static constexpr int CTILE_BYTES = (CBOX_BYTES + 127) / 128 * 128;
    static constexpr int NC = 4;
    static_assert(CW >= CWN + VEC - 1, "coarse tile too narrow");
    static_assert(PLANE_BYTES % 128 == 0 && BOX_BYTES % 128 == 0 && (BW * ES) % 128 == 0, "TMA destinations are 128-B aligned");
};

// One Jacobi stage of the 2-D form on a pack (r02): out = v + w_p (((pv + nx) + (xm + xp)) - 4 v) + h^2 g), Eq. 3 in the
// order of DESIGN.md R14, with the Dirichlet condition as the per-node multiplier w_p in {w/4, 0} (v is 0 there, so
// v + 0 t = 0) instead of a select.  fp32: packed pairs (FADD2 / FFMA2), the same bits at half the issue slots.
template <class T>
__device__ __forceinline__ Pack<T> jacobi_pack2d(const Pack<T>& pv, const Pack<T>& cu, const Pack<T>& nx, const Pack<T>& gv, T vl,
                                                 T vr, const Pack<T>& wpm, const Coef<T>& cf) {
    constexpr int VEC = 16 / int(sizeof(T));
    Pack<T> out;
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
        const T vc = cu.v[j];
        const T xm = j == 0 ? vl : cu.v[j - 1 < 0 ? 0 : j - 1];
        const T xp = j == VEC - 1 ? vr : cu.v[j + 1 > VEC - 1 ? VEC - 1 : j + 1];
        T sm = pv.v[j] + nx.v[j];
        sm += xm + xp;
        T t = fma_rn(-cf.twod, vc, sm);
        t = fma_rn(cf.h2, gv.v[j], t);
        out.v[j] = fma_rn(wpm.v[j], t, vc);
    }
    return out;
}
__device__ __forceinline__ Pack<float> jacobi_pack2d(const Pack<float>& pv, const Pack<float>& cu, const Pack<float>& nx,
                                                     const Pack<float>& gv, float vl, float vr, const Pack<float>& wpm,
                                                     const Coef<float>& cf) {
    const F2 ntd = f2_make(-cf.twod, -cf.twod), h2 = f2_make(cf.h2, cf.h2);
    const float xs[4] = {vl + cu.v[1], cu.v[0] + cu.v[2], cu.v[1] + cu.v[3], cu.v[2] + vr};
    Pack<float> out;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const F2 c2 = f2_make(cu.v[2 * h], cu.v[2 * h + 1]);
        F2 sm = f2_add(f2_make(pv.v[2 * h], pv.v[2 * h + 1]), f2_make(nx.v[2 * h], nx.v[2 * h + 1]));
        sm = f2_add(sm, f2_make(xs[2 * h], xs[2 * h + 1]));
        F2 t = f2_fma(ntd, c2, sm);
        t = f2_fma(h2, f2_make(gv.v[2 * h], gv.v[2 * h + 1]), t);
        f2_get(f2_fma(f2_make(wpm.v[2 * h], wpm.v[2 * h + 1]), t, c2), out.v[2 * h], out.v[2 * h + 1]);
    }
    return out;
}

template <class T, int ND, int NS, bool INTERP>
__host__ __device__ constexpr int visit_smem_bytes() {
    using TL = VisitTile<T, ND, NS>;
    return TL::NGR * TL::BOX_BYTES +
           (INTERP ? TL::NC * 2 * TL::CTILE_BYTES + NS * 2 * TL::PLANE_BYTES
                   : TL::NIN * TL::PLANE_BYTES + (NS - 1) * 2 * TL::PLANE_BYTES) + 128;
}

// tm_in : PLAIN: v^0 of this level, box {TXN, PY, 1};  INTERP: e_c of level c = t+1, box {CW, CR, 1}
// tm_ac : INTERP: a_c, same box;  tm_g : g of this level, box {TXN, PY, 1}
// o0 / o1 / o2 : v^NS, v^{NS-1}, v^{NS-2} (each may be null);  a, a_assign, d0, v0, u : as k_relax
// grid = (x tiles of OX, y tiles of OY, z chunks of mchunk interior planes);  2-D: (x tiles, y chunks)
// ("z" / "plane" below = the marching axis: z in 3-D, y in 2-D)
// BOOK: the visit of a level >= 1 (S3e bookkeeping, v^{NS-1} / v^{NS-2} stored, no u); otherwise a level-0
// visit (u optional, nothing else) — two compiled variants so that neither carries the other's registers.
// CTAs per SM the register allocation aims at: 3-D one 512-thread CTA; 2-D (160 threads) four level-0 CTAs
// (<= 96 registers) or three with the S3e bookkeeping
template <int ND, bool BOOK>
__host__ __device__ constexpr int visit_ctas() { return ND == 3 ? 1 : (BOOK ? 3 : 4); }

template <class T, int ND, int NS, bool INTERP, bool BOOK>
__global__ void __launch_bounds__(VisitTile<T, ND, NS>::NT, visit_ctas<ND, BOOK>())
k_visit(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_ac,
         const __grid_constant__ CUtensorMap tm_g, LevelGeom g, Coef<T> cf, T* __restrict__ o0,
         T* __restrict__ o1, T* __restrict__ o2, T* __restrict__ a, int a_assign, const T* __restrict__ d0,
         const T* __restrict__ v0, T* __restrict__ u, int mchunk) {
    pdl_start();
    using TL = VisitTile<T, ND, NS>;
    constexpr int VEC = TL::VEC, RS = TL::RS;
    const int tid = threadIdx.x, px = tid % TL::PX, py = tid / TL::PX;
    const int NM = ND == 3 ? g.nz : g.ny;
    const long long mstride = ND == 3 ? g.pp : (long long)g.px;
    const int x0 = blockIdx.x * TL::OX, y0 = ND == 3 ? blockIdx.y * TL::OY : 0;
    const int ms = 1 + (ND == 3 ? blockIdx.z : blockIdx.y) * mchunk;
    const int me = min(ms + mchunk, NM - 1);
    if (ms >= me) return;
    const int zs = ms - NS;                                        // first plane of stage 0
    const int nsteps = me - ms + 2 * NS;                           // one stage-0 plane per step
    const int Zc0 = zs >> 1;                                       // first coarse plane (floor)
    const int ncz = ((me + NS) >> 1) - Zc0 + 1;

    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    __shared__ uint64_t fbar[TL::NIN], gbar[TL::NGR], cbar[TL::NC];
    auto gs = [&](int st) { return reinterpret_cast<T*>(smem + st * TL::BOX_BYTES); };
    unsigned char* cbase = smem + TL::NGR * TL::BOX_BYTES;         // PLAIN: v ring;  INTERP: coarse ring
    auto vring = [&](int st) { return reinterpret_cast<T*>(cbase + st * TL::PLANE_BYTES); };
    auto ce = [&](int st) { return reinterpret_cast<T*>(cbase + (2 * st) * TL::CTILE_BYTES); };
    auto ca = [&](int st) { return reinterpret_cast<T*>(cbase + (2 * st + 1) * TL::CTILE_BYTES); };
    unsigned char* sbase = cbase + (INTERP ? TL::NC * 2 * TL::CTILE_BYTES : TL::NIN * TL::PLANE_BYTES);
    auto buf = [&](int s, int slot) {                              // plane published by stage s
        return reinterpret_cast<T*>(sbase + ((INTERP ? s : s - 1) * 2 + slot) * TL::PLANE_BYTES);
    };

    if (tid == 0) {
        for (int s = 0; s < TL::NIN; ++s) mbar_init(&fbar[s], 1);
        for (int s = 0; s < TL::NGR; ++s) mbar_init(&gbar[s], 1);
        for (int s = 0; s < TL::NC; ++s) mbar_init(&cbar[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    const int Xc = (x0 - TL::HX) / 2;                              // x0 - HX is even
    const int Xa = Xc - (Xc & (VEC - 1));                          // coarse box start, 16-B aligned
    const int Yc = (y0 - TL::HY) >> 1;
    auto issue_f = [&](int q) {                                    // fine plane zs+q: (v^0 and) g
        const int st = q & (TL::NIN - 1), sg = q & (TL::NGR - 1), p = zs + q;
        if (!INTERP) {
            mbar_arrive_expect_tx(&fbar[st], TL::BOX_BYTES);
            if (ND == 3) tma_load_3d(vring(st) + TL::ROFF, &tm_in, &fbar[st], x0 - TL::HX, y0 - TL::HY, p);
            else
                for (int b = 0; b < TL::TXN / TL::BW; ++b)
                    tma_load_2d(vring(st) + TL::ROFF + b * TL::BW, &tm_in, &fbar[st], x0 - TL::HX + b * TL::BW, p);
        }
        mbar_arrive_expect_tx(&gbar[sg], TL::BOX_BYTES);
        if (ND == 3) tma_load_3d(gs(sg), &tm_g, &gbar[sg], x0 - TL::HX, y0 - TL::HY, p);
        else
            for (int b = 0; b < TL::TXN / TL::BW; ++b)
                tma_load_2d(gs(sg) + b * TL::BW, &tm_g, &gbar[sg], x0 - TL::HX + b * TL::BW, p);
    };
    auto issue_c = [&](int zc) {                                   // coarse plane Zc0+zc of e_c and a_c
        const int st = zc & (TL::NC - 1);
        mbar_arrive_expect_tx(&cbar[st], 2 * TL::CBOX_BYTES);
        if (ND == 3) {
            tma_load_3d(ce(st), &tm_in, &cbar[st], Xa, Yc, Zc0 + zc);
            tma_load_3d(ca(st), &tm_ac, &cbar[st], Xa, Yc, Zc0 + zc);
        } else {
            for (int b = 0; b < TL::NCB; ++b) {
                tma_load_2d(ce(st) + b * TL::CBW, &tm_in, &cbar[st], Xa + b * TL::CBW, Zc0 + zc);
                tma_load_2d(ca(st) + b * TL::CBW, &tm_ac, &cbar[st], Xa + b * TL::CBW, Zc0 + zc);
            }
        }
    };
    if (tid == 0) {
        if (INTERP)
            for (int zc = 0; zc < TL::NC && zc < ncz; ++zc) issue_c(zc);
        for (int q = 0; q < TL::NIN - 1 && q < nsteps; ++q) issue_f(q);
    }

    // ---- this thread's pack: nodes x .. x+VEC-1 of row y ----
    const int x = x0 - TL::HX + px * VEC;
    const int y = y0 - TL::HY + py;                                // 2-D: 0, unused
    const int off = TL::ROFF + py * RS + px * VEC;                 // in a padded plane
    const int goff = py * RS + px * VEC;
    const bool row_int = ND == 2 || (y > 0 && y < g.ny - 1);
    bool xin[VEC];
#pragma unroll
    for (int j = 0; j < VEC; ++j) xin[j] = row_int && (x + j > 0) && (x + j < g.nx - 1);
    Pack<T> wpm;                                                   // 2-D: Eq. 3's w_p, 0 off the interior
#pragma unroll
    for (int j = 0; j < VEC; ++j) wpm.v[j] = xin[j] ? cf.wp : T(0);
    const bool own = px * VEC >= TL::HX && px * VEC < TL::HX + TL::OX && x < g.nx &&
                     (ND == 2 || (py >= TL::HY && py < TL::HY + TL::OY && y < g.ny));
    // INTERP: my first coarse node inside a coarse tile
    const int yl = ND == 3 ? (y >> 1) - Yc : 0;
    const bool yodd = ND == 3 && (y & 1);
    const int coff = yl * TL::CW + (Xc - Xa) + px * (VEC / 2);

    // S3a in registers: the pack of v^0 at fine plane z from the coarse planes z>>1 and (z+1)>>1;
    // summation order as homg_first.cuh / the oracle: rows (z lo, y lo), (z lo, y hi), (z hi, y lo), (z hi, y hi)
    auto produce = [&](const int z) -> Pack<T> {
        constexpr int NCV = VEC / 2 + 1;
        const bool zodd = z & 1;
        const int zlo = (z >> 1) - Zc0, zhi = ((z + 1) >> 1) - Zc0;
        mbar_wait(&cbar[zlo & (TL::NC - 1)], (zlo / TL::NC) & 1);
        if (zodd) mbar_wait(&cbar[zhi & (TL::NC - 1)], (zhi / TL::NC) & 1);
        const T* A0 = ca(zlo & (TL::NC - 1)) + coff;
        const T* A1 = ca(zhi & (TL::NC - 1)) + coff;
        const T* E0 = ce(zlo & (TL::NC - 1)) + coff;
        T acc[VEC];
        auto addrow = [&](const T* rp, const bool first) {
            T c[NCV];
            if (VEC == 4) {
                const HalfPack<T> h = *reinterpret_cast<const HalfPack<T>*>(rp);
                c[0] = h.v[0]; c[1] = h.v[1]; c[NCV - 1] = rp[NCV - 1];
            } else {
#pragma unroll
                for (int i = 0; i < NCV; ++i) c[i] = rp[i];
            }
#pragma unroll
            for (int j = 0; j < VEC; ++j) {
                if (j & 1) { acc[j] = first ? c[j >> 1] : acc[j] + c[j >> 1]; acc[j] += c[(j >> 1) + 1]; }
                else acc[j] = first ? c[j >> 1] : acc[j] + c[j >> 1];
            }
        };
        addrow(A0, true);
        if (yodd) addrow(A0 + TL::CW, false);
        if (zodd) {
            addrow(A1, false);
            if (yodd) addrow(A1 + TL::CW, false);
        }
        const T wzy = (zodd && yodd) ? T(0.25) : ((zodd || yodd) ? T(0.5) : T(1));
        const bool coin = !zodd && !yodd;
        Pack<T> out;
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
            if (j & 1) out.v[j] = (T(0.5) * wzy) * acc[j];
            else out.v[j] = coin ? E0[j >> 1] : wzy * acc[j];
        }
        return out;
    };

    // register state: own column of every stage input (previous and current plane), g of the stages
    // g of a plane read once and carried down the stages in registers: measured slower in this kernel (the 12 registers it
    // costs spill at the 96 that four CTAs per SM leave: level-0 visit of cfg3 259 -> 275 us) — kept switchable, off
#ifndef HOMG_VISIT2D_G_CHAIN
#define HOMG_VISIT2D_G_CHAIN 0
#endif
    constexpr bool G_CHAIN = ND == 2 && HOMG_VISIT2D_G_CHAIN;
    Pack<T> P[NS], C[NS];
    Pack<T> Gh[NS - 1];
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
            P[s].v[j] = T(0); C[s].v[j] = T(0);
            if (s < NS - 1) Gh[s].v[j] = T(0);
        }

    // address of (x, y) in the plane the LAST stage produces at step q: z = zs + q - NS
    long long cF = (long long)(zs - NS) * mstride + (ND == 3 ? (long long)y * g.px : 0) + x;

    // STEADY: the pipeline is full and every stage's plane is interior — no range checks
    auto step = [&](auto KC, auto SD, const int q) {
        constexpr int W = decltype(KC)::value, R = W ^ 1;          // stage-buffer slots: written now / read now
        constexpr bool STEADY = decltype(SD)::value;
        const int K = q & (TL::NIN - 1), SC = (q - 1) & (TL::NIN - 1);   // v ring slots of planes z0, z0-1
        const int z0 = zs + q;
        // ---- stage 0: the pack of v^0 at plane z0 ----
        Pack<T> nx;
        if (INTERP) {
            nx = produce(z0);
            if (ND == 3) *reinterpret_cast<Pack<T>*>(buf(0, W) + off) = nx;
            else {                                                 // 2-D: only the x neighbours across warp borders are read back
                if ((tid & 31) == 0) buf(0, W)[off] = nx.v[0];
                if ((tid & 31) == 31) buf(0, W)[off + VEC - 1] = nx.v[VEC - 1];
            }
        } else {
            mbar_wait(&fbar[K], (q / TL::NIN) & 1);
            nx = *reinterpret_cast<const Pack<T>*>(vring(K) + off);
        }
        // u of the plane the last stage produces in this step: loaded now, used after the NS stages,
        // so that its HBM latency hides behind the arithmetic
        const bool fin = own && (STEADY || q >= 2 * NS);
        Pack<T> uu;
        if (!BOOK && fin && u) uu = *reinterpret_cast<const Pack<T>*>(u + cF);
        static_assert(!(INTERP && BOOK), "interpolate+correct is fused on level 0 only");
        if (BOOK && fin && a) {                                    // S3e operands: into L1 now (no registers), read after the stages
            asm volatile("prefetch.global.L1 [%0];" ::"l"(v0 + cF));
            if (d0) asm volatile("prefetch.global.L1 [%0];" ::"l"(d0 + cF));
            if (!a_assign) asm volatile("prefetch.global.L1 [%0];" ::"l"(a + cF));
        }
        // stage s reads g of plane z0-s from the g ring; plane z0-1 is new in this step
        if (STEADY || q >= 1) mbar_wait(&gbar[(q - 1) & (TL::NGR - 1)], ((q - 1) / TL::NGR) & 1);
        // shared-memory operands of a stage (y neighbours, g; 2-D: the x neighbours across warp borders).
        // They were published in the previous step, so the operands of stage s+1 are fetched BEFORE stage s
        // computes and stores: the compiler cannot move a load above a shared store by itself.
        auto fetch = [&](const int s, Pack<T>& dn, Pack<T>& up, Pack<T>& gv, T& el, T& er) {
            const T* ctr = (s == 1 && !INTERP) ? vring(SC) : buf(s - 1, R);
            if (ND == 3) {
                dn = *reinterpret_cast<const Pack<T>*>(ctr + off - RS);
                up = *reinterpret_cast<const Pack<T>*>(ctr + off + RS);
            } else {
                if ((tid & 31) == 0) el = ctr[off - 1];
                if ((tid & 31) == 31) er = ctr[off + VEC];
            }
            if (!G_CHAIN || s == 1) gv = *reinterpret_cast<const Pack<T>*>(gs((q - s) & (TL::NGR - 1)) + goff);
            else gv = Gh[s - 2 < 0 ? 0 : s - 2];                   // read at stage 1 of an earlier step
        };
        // (3-D: one CTA of 512 threads per SM leaves 128 registers per thread; fetching ahead spills there)
        constexpr bool AHEAD = ND == 2 || !BOOK;
        Pack<T> dnN, upN, gvN;
        T elN = T(0), erN = T(0);
        if (AHEAD) fetch(1, dnN, upN, gvN, elN, erN);
        Pack<T> g1 = gvN;                                          // 2-D: g of plane z0-1, enters the chain after the stages
#pragma unroll
        for (int s = 1; s <= NS; ++s) {
            // stage s: plane z0-s of v^s from v^{s-1}: P (z0-s-1), C (z0-s), nx (z0-s+1)
            if (!AHEAD) { fetch(s, dnN, upN, gvN, elN, erN); if (s == 1) g1 = gvN; }
            const Pack<T> dn = dnN, up = upN, gv = gvN;
            const T el = elN, er = erN;
            if (AHEAD && s < NS) fetch(s + 1, dnN, upN, gvN, elN, erN);
            const Pack<T> cu = C[s - 1], pv = P[s - 1];
            T vl = __shfl_up_sync(0xffffffffu, cu.v[VEC - 1], 1);
            T vr = __shfl_down_sync(0xffffffffu, cu.v[0], 1);
            if (ND == 2) {                                         // a row spans several warps
                if ((tid & 31) == 0) vl = el;
                if ((tid & 31) == 31) vr = er;
            }
            const int z = z0 - s;
            const bool zin = STEADY || (z > 0 && z < NM - 1);
            Pack<T> out;
            if (ND == 2) {
                out = jacobi_pack2d(pv, cu, nx, gv, vl, vr, wpm, cf);
            } else {
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    const T vc = cu.v[j];
                    const T xm = j == 0 ? vl : cu.v[j - 1 < 0 ? 0 : j - 1];
                    const T xp = j == VEC - 1 ? vr : cu.v[j + 1 > VEC - 1 ? VEC - 1 : j + 1];
                    T sm = pv.v[j] + nx.v[j];
                    sm += dn.v[j] + up.v[j];
                    sm += xm + xp;
                    out.v[j] = xin[j] ? jacobi_eq3(vc, sm, gv.v[j], cf) : T(0);
                }
            }
            if (!zin) {                                            // Dirichlet planes z = 0, nz-1 (and beyond)
#pragma unroll
                for (int j = 0; j < VEC; ++j) out.v[j] = T(0);
            }
            if (s < NS) {
                if (ND == 3) *reinterpret_cast<Pack<T>*>(buf(s, W) + off) = out;
                else {
                    if ((tid & 31) == 0) buf(s, W)[off] = out.v[0];
                    if ((tid & 31) == 31) buf(s, W)[off + VEC - 1] = out.v[VEC - 1];
                }
            }
            if (BOOK && s == NS - 2 && s >= 1 && o2 != nullptr && own && (STEADY || (q >= 2 * NS - 2 && q <= nsteps - 3)))
                *reinterpret_cast<Pack<T>*>(o2 + cF + 2 * mstride) = out;
            if (BOOK && s == NS - 1 && s >= 1 && o1 != nullptr && own && (STEADY || (q >= 2 * NS - 1 && q <= nsteps - 2)))
                *reinterpret_cast<Pack<T>*>(o1 + cF + mstride) = out;
            if (s == NS && fin) {
                if (o0) *reinterpret_cast<Pack<T>*>(o0 + cF) = out;
                if (BOOK && a) {                                   // S3e: a (+)= d0 + v^{NS-1} - v^0
                    Pack<T> dd, vv = *reinterpret_cast<const Pack<T>*>(v0 + cF), aa;
                    if (d0) dd = *reinterpret_cast<const Pack<T>*>(d0 + cF);
                    if (!a_assign) aa = *reinterpret_cast<const Pack<T>*>(a + cF);
#pragma unroll
                    for (int j = 0; j < VEC; ++j) {
                        const T Dq = ((d0 ? dd.v[j] : T(0)) + cu.v[j]) - vv.v[j];
                        aa.v[j] = a_assign ? Dq : aa.v[j] + Dq;
                    }
                    *reinterpret_cast<Pack<T>*>(a + cF) = aa;
                }
                if (!BOOK && u) {                                  // S4: u += v^NS
#pragma unroll
                    for (int j = 0; j < VEC; ++j) uu.v[j] += out.v[j];
                    *reinterpret_cast<Pack<T>*>(u + cF) = uu;
                }
            }
            P[s - 1] = cu; C[s - 1] = nx; nx = out;
        }
        if (G_CHAIN) {
#pragma unroll
            for (int s = NS - 2; s >= 1; --s) Gh[s] = Gh[s - 1];
            Gh[0] = g1;
        }
        __syncthreads();
        if (tid == 0) {
            if (q + TL::NIN - 1 < nsteps) issue_f(q + TL::NIN - 1);
            if (INTERP && (z0 & 1)) {                              // coarse plane z0>>1 is dead now
                const int zc = (z0 >> 1) - Zc0 + TL::NC;
                if (zc < ncz) issue_c(zc);
            }
        }
        cF += mstride;
    };
    using I0 = std::integral_constant<int, 0>;
    using I1 = std::integral_constant<int, 1>;
    for (int q = 0; q < nsteps; q += 2) {
        // steps q and q+1 are steady when all their stores are due and planes z0-NS .. z0-1 are interior
        const bool steady = q >= 2 * NS && q + 1 <= nsteps - 3 && zs + q - NS >= 1 && zs + q <= NM - 2;
        if (steady) {
            step(I0{}, std::true_type{}, q);
            step(I1{}, std::true_type{}, q + 1);
        } else {
            step(I0{}, std::false_type{}, q);
            if (q + 1 < nsteps) step(I1{}, std::false_type{}, q + 1);
        }
    }
}

}  // namespace homg
