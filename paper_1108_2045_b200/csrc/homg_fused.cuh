// homg_fused.cuh — tiled sm_100a kernels for the LARGE levels of the HOMG cycle.
//
// Common scheme (north_star items 2-3): a CTA of 256 threads owns an x/y tile and marches along the
// slowest axis (z in 3-D, y in 2-D).  Every plane of the tile (plus halo) is brought into a 4-stage
// shared-memory ring by TMA (cp.async.bulk.tensor, completion on an mbarrier), three planes ahead of
// the one being computed; out-of-range halo elements arrive as 0, which is the Dirichlet value.
// Threads hold VEC = 16 B / sizeof(T) consecutive x nodes each (LDS.128 / STG.128) and keep the
// previous / current / next plane of their own nodes in registers (register blocking along the
// slowest axis), so shared memory is read only for the in-plane neighbours.
//
// The arithmetic is the expression tree of homg_kernels.cuh (R14) — results are bit-identical
// to the generic kernels and to the oracle.
#pragma once
#include <type_traits>

#include "homg_kernels.cuh"
#include "homg_tma.cuh"

namespace homg {

template <class T>
struct alignas(16) Pack {
    T v[16 / sizeof(T)];
};

template <class T>
struct alignas(2 * sizeof(T)) HalfPack {
    T v[2];
};

// sm_100a packed fp32 pairs: add / fma .rn.f32x2 (SASS FADD2 / FFMA2) are two IEEE round-to-nearest operations per
// instruction — the bits of the scalar form at half the issue slots (used by K_visit, 2-D and 3-D)
struct F2 { unsigned long long b; };
__device__ __forceinline__ F2 f2_make(float lo, float hi) { F2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.b) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void f2_get(F2 a, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.b)); }
__device__ __forceinline__ F2 f2_add(F2 a, F2 b) { F2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.b) : "l"(a.b), "l"(b.b)); return r; }
__device__ __forceinline__ F2 f2_fma(F2 a, F2 b, F2 c) { F2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.b) : "l"(a.b), "l"(b.b), "l"(c.b)); return r; }

// x / D for a per-level constant D with rD = RN(1/D) precomputed on the host: q = RN(x rD),
// r = x - q D (exact in one FMA), result RN(q + r rD).  By Markstein's theorem this is the correctly
// rounded quotient, i.e. bit-identical to the IEEE division the generic kernels and the oracle
// perform, at 3 instructions instead of a division sequence (tests: tiled == generic bitwise).
__device__ __forceinline__ float div_const(float x, float D, float rD) {
    const float q = x * rD;
    return __fmaf_rn(__fmaf_rn(-q, D, x), rD, q);
}
__device__ __forceinline__ double div_const(double x, double D, double rD) {
    const double q = x * rD;
    return __fma_rn(__fma_rn(-q, D, x), rD, q);
}

template <class T, int ND>
struct Tile {
    static constexpr int VEC = 16 / int(sizeof(T));
    static constexpr int WY = ND == 3 ? 8 : 1;           // warps along y
    static constexpr int WX = 8 / WY;                    // warps (segments) along x
    static constexpr int SEG = 32 * VEC;                 // x nodes per warp
    static constexpr int TX = WX * SEG, TY = WY;         // nodes per CTA and plane
    static constexpr int VW = SEG + 2 * VEC;             // halo'd row width (one TMA box row)
    static constexpr int VROWS = ND == 3 ? TY + 2 : WX;  // rows of the halo'd tile in shared memory
    // 3-D: one box {VW, TY+2, 1}, rows contiguous.  2-D: WX boxes {VW, 1}, each 128-B aligned.
    static constexpr int VRS = ND == 3 ? VW : ((VW * int(sizeof(T)) + 127) / 128 * 128) / int(sizeof(T));
    static constexpr int VBOX_BYTES = VROWS * VW * int(sizeof(T));             // bytes TMA delivers
    static constexpr int VTILE_BYTES = (VROWS * VRS * int(sizeof(T)) + 127) / 128 * 128;
    static constexpr int GROWS = ND == 3 ? TY : WX;
    static constexpr int GBOX_BYTES = GROWS * SEG * int(sizeof(T));            // = tile bytes (128-B multiple)
    static constexpr int NST = 4;
};

template <class T, int ND, bool VAR>
__host__ __device__ constexpr int relax_stage_bytes() {
    return Tile<T, ND>::VTILE_BYTES + Tile<T, ND>::GBOX_BYTES;
}
template <class T, int ND, bool VAR>
__host__ __device__ constexpr int relax_smem_bytes() {
    return relax_stage_bytes<T, ND, VAR>() * Tile<T, ND>::NST + 128;
}

// S3d (+S3e, +S4): one damped-Jacobi sweep  vout = vin + w (g - A vin)/D  on a large level.
//   tmv / tmg : tensor maps of vin and g of this level;  kf : face coefficients (VAR), read straight
//   from global memory as coalesced 16-byte packs (own pack of fz / fy / fx, the y-1 row of fy, one scalar of fx)
//   a, a_assign, d0, v0, u : the optional epilogues of k_relax (same meaning)
//   vout may be null when u is given (last sweep of the cycle: e_0 is dead after u += e_0)
//   mchunk : interior planes per CTA along the marching axis
// grid = (x tiles, y tiles, chunks) in 3-D, (x tiles, chunks) in 2-D.      (Eq.2-3)
template <class T, int ND, bool VAR>
__global__ void __launch_bounds__(256)
k_relax_tma(const __grid_constant__ CUtensorMap tmv, const __grid_constant__ CUtensorMap tmg,
            Faces<T> kf, LevelGeom g, Coef<T> cf, T* __restrict__ vout,
            T* __restrict__ a, int a_assign, const T* __restrict__ d0, const T* __restrict__ v0,
            T* __restrict__ u, int mchunk) {
    pdl_start();
    using TL = Tile<T, ND>;
    constexpr int VEC = TL::VEC;
    constexpr int STAGE = relax_stage_bytes<T, ND, VAR>();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wx = warp % TL::WX, wy = warp / TL::WX;
    const int NM = ND == 3 ? g.nz : g.ny;
    const long long mstride = ND == 3 ? g.pp : (long long)g.px;
    const int x0 = blockIdx.x * TL::TX;
    const int y0 = ND == 3 ? blockIdx.y * TL::TY : 0;
    const int chunk = ND == 3 ? blockIdx.z : blockIdx.y;
    const int ms = 1 + chunk * mchunk;
    const int me = min(ms + mchunk, NM - 1);
    if (ms >= me) return;
    const int count = me - ms + 2;                       // planes ms-1 .. me

    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);   // keeps the shared address space
    __shared__ uint64_t bars[TL::NST];
    auto vs = [&](int st) { return reinterpret_cast<T*>(smem + st * STAGE); };
    auto gs = [&](int st) { return reinterpret_cast<T*>(smem + st * STAGE + TL::VTILE_BYTES); };

    if (tid == 0) {
        for (int s = 0; s < TL::NST; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int i) {                            // relative plane i = absolute ms-1+i
        const int st = i & (TL::NST - 1), p = ms - 1 + i;
        const bool wantg = i >= 1 && i <= count - 2;
        mbar_arrive_expect_tx(&bars[st], TL::VBOX_BYTES + (wantg ? TL::GBOX_BYTES : 0));
        if (ND == 3) {
            tma_load_3d(vs(st), &tmv, &bars[st], x0 - VEC, y0 - 1, p);
            if (wantg) tma_load_3d(gs(st), &tmg, &bars[st], x0, y0, p);
        } else {
            for (int w = 0; w < TL::WX; ++w) {
                tma_load_2d(vs(st) + w * TL::VRS, &tmv, &bars[st], x0 + w * TL::SEG - VEC, p);
                if (wantg) tma_load_2d(gs(st) + w * TL::SEG, &tmg, &bars[st], x0 + w * TL::SEG, p);
            }
        }
    };

    // this thread's nodes: x .. x+VEC-1 of row y; its row inside the halo'd tile
    const int x = x0 + wx * TL::SEG + lane * VEC;
    const int y = ND == 3 ? y0 + wy : 0;
    const int vrow = ND == 3 ? wy + 1 : wx;
    const int voff = vrow * TL::VRS + VEC + lane * VEC;  // centre pack inside a v / k tile
    const int goff = (ND == 3 ? wy : wx) * TL::SEG + lane * VEC;
    const bool row_ok = x < g.nx && (ND == 2 || y < g.ny);
    const bool row_int = ND == 2 || (y > 0 && y < g.ny - 1);
    bool xin[VEC];
#pragma unroll
    for (int j = 0; j < VEC; ++j) xin[j] = row_int && (x + j > 0) && (x + j < g.nx - 1);

    if (tid == 0)
        for (int i = 0; i < TL::NST && i < count; ++i) issue(i);

    Pack<T> prv, cur, nxt;
    mbar_wait(&bars[0], 0);
    prv = *reinterpret_cast<const Pack<T>*>(vs(0) + voff);
    mbar_wait(&bars[1], 0);
    cur = *reinterpret_cast<const Pack<T>*>(vs(1) + voff);
    __syncthreads();
    if (tid == 0 && TL::NST < count) issue(TL::NST);

    long long c = (long long)ms * mstride + (ND == 3 ? (long long)y * g.px : 0) + x;
    // VAR: faces of this thread's nodes; the z- face of a plane is the z+ face of the one before
    const bool kok = VAR && row_ok && row_int;
    Pack<T> fzm, nfz, nfym, nfyp, nfx;
    T nfxl = T(0);
    auto fetch_faces = [&](const long long cc) {
        nfz = *reinterpret_cast<const Pack<T>*>(kf.z + cc);
        nfym = *reinterpret_cast<const Pack<T>*>(kf.y + cc - g.px);
        nfyp = *reinterpret_cast<const Pack<T>*>(kf.y + cc);
        nfx = *reinterpret_cast<const Pack<T>*>(kf.x + cc);
        if (x > 0) nfxl = kf.x[cc - 1];
    };
    if (kok) {
        fzm = *reinterpret_cast<const Pack<T>*>(kf.z + c - mstride);
        fetch_faces(c);
    }
    // one plane; K = (i-1) mod 4 is a compile-time constant so that every stage address is an immediate
    auto step = [&](auto KC, const int i) {
        constexpr int K = decltype(KC)::value;
        constexpr int sn = (K + 2) & (TL::NST - 1), sc = (K + 1) & (TL::NST - 1);
        // faces of this plane were fetched one step ago; those of the next plane (it exists: z+1 <= NM-1) now
        const Pack<T> fzp = nfz, fym = nfym, fyp = nfyp, fxp = nfx;
        const T fxl = nfxl;
        if (kok) fetch_faces(c + mstride);
        // operands of the NEXT plane's epilogues (S4: u; S3e: v0, d0, a) into L1 now (no registers)
        if (row_ok) {
            if (u) asm volatile("prefetch.global.L1 [%0];" ::"l"(u + c + mstride));
            if (a) {
                asm volatile("prefetch.global.L1 [%0];" ::"l"(v0 + c + mstride));
                if (d0) asm volatile("prefetch.global.L1 [%0];" ::"l"(d0 + c + mstride));
                if (!a_assign) asm volatile("prefetch.global.L1 [%0];" ::"l"(a + c + mstride));
            }
        }
        mbar_wait(&bars[sn], ((i + 1) / TL::NST) & 1);
        nxt = *reinterpret_cast<const Pack<T>*>(vs(sn) + voff);
        const T* vt = vs(sc);
        Pack<T> dn, up;
        if (ND == 3) {
            dn = *reinterpret_cast<const Pack<T>*>(vt + voff - TL::VRS);
            up = *reinterpret_cast<const Pack<T>*>(vt + voff + TL::VRS);
        }
        const T vl = vt[voff - 1], vr = vt[voff + VEC];
        const Pack<T> gv = *reinterpret_cast<const Pack<T>*>(gs(sc) + goff);
        Pack<T> out;
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
            const T vc = cur.v[j];
            const T xm = j == 0 ? vl : cur.v[j - 1 < 0 ? 0 : j - 1];
            const T xp = j == VEC - 1 ? vr : cur.v[j + 1 > VEC - 1 ? VEC - 1 : j + 1];
            T Av = T(0), D = T(1), eq3 = T(0);
            if (!VAR) {
                T s = prv.v[j] + nxt.v[j];
                if (ND == 3) s += dn.v[j] + up.v[j];
                s += xm + xp;
                eq3 = jacobi_eq3(vc, s, gv.v[j], cf);
            } else {
                const T fxm = j == 0 ? fxl : fxp.v[j - 1 < 0 ? 0 : j - 1];
                T acc = T(0), ds = T(0);
                acc += fzm.v[j] * (vc - prv.v[j]); ds += fzm.v[j];
                acc += fzp.v[j] * (vc - nxt.v[j]); ds += fzp.v[j];
                if (ND == 3) {
                    acc += fym.v[j] * (vc - dn.v[j]); ds += fym.v[j];
                    acc += fyp.v[j] * (vc - up.v[j]); ds += fyp.v[j];
                }
                acc += fxm * (vc - xm); ds += fxm;
                acc += fxp.v[j] * (vc - xp); ds += fxp.v[j];
                Av = acc * cf.ih2;
                D = ds * cf.ih2;
            }
            out.v[j] = xin[j] ? (VAR ? vc + cf.w * (gv.v[j] - Av) / D : eq3) : T(0);
        }
        if (row_ok) {
            if (vout) *reinterpret_cast<Pack<T>*>(vout + c) = out;
            if (a) {
                Pack<T> dd, vv = *reinterpret_cast<const Pack<T>*>(v0 + c), aa;
                if (d0) dd = *reinterpret_cast<const Pack<T>*>(d0 + c);
                if (!a_assign) aa = *reinterpret_cast<const Pack<T>*>(a + c);
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    const T Dq = ((d0 ? dd.v[j] : T(0)) + cur.v[j]) - vv.v[j];
                    aa.v[j] = a_assign ? Dq : aa.v[j] + Dq;
                }
                *reinterpret_cast<Pack<T>*>(a + c) = aa;
            }
            if (u) {
                Pack<T> uu = *reinterpret_cast<const Pack<T>*>(u + c);
#pragma unroll
                for (int j = 0; j < VEC; ++j) uu.v[j] += out.v[j];
                *reinterpret_cast<Pack<T>*>(u + c) = uu;
            }
        }
        __syncthreads();
        if (tid == 0 && i + TL::NST < count) issue(i + TL::NST);
        prv = cur; cur = nxt;
        if (VAR) fzm = fzp;
        c += mstride;
    };
    for (int i = 1; i <= count - 2; i += 4) {
        step(std::integral_constant<int, 0>{}, i);
        if (i + 1 > count - 2) break;
        step(std::integral_constant<int, 1>{}, i + 1);
        if (i + 2 > count - 2) break;
        step(std::integral_constant<int, 2>{}, i + 2);
        if (i + 3 > count - 2) break;
        step(std::integral_constant<int, 3>{}, i + 3);
    }
}


// ---------------------------------------------------------------------------------------------
// K_res: fused residual + ||r||^2 partial + first full-weighting restriction (S1 + S2 first step + S5).
//
// The CTA computes r = f - A u on an r-tile that is one node wider than what it owns, on the low
// side of every axis (full weighting of the coarse nodes of a tile needs r at 2I-1).  3-D: a row of
// the r-tile is 33 packs: pack 0 is the recomputed halo pack [x0-VEC, x0), packs 1..32 are owned, so
// a tile owns 32*VEC x 8 nodes per plane (power-of-two widths: 2^k+1 grids tile without a mostly
// empty last tile).  Warps 0..8 = fine rows y0-1 .. y0+7 (row 0 is the recomputed halo row), lane l =
// pack l+1; warp 9 computes the 9 halo packs (lane l = row l; its other lanes repeat row 0).  2-D: 8
// warps = 8 x-segments of one row, lane 0 of each its private halo pack.  Every thread runs the same code.  The last four r planes stay in shared memory; after
// an odd plane z = 2Z+1 the CTA writes the coarse plane Z (27 / 9 terms in the oracle's order).
// A chunk [ms, me) of the marching axis (ms odd, even length) recomputes plane `me` for the same
// reason.  r may be null (norm only); gc may be null (no restriction).
//
template <class T, int ND>
struct ResTile {
    static constexpr int VEC = 16 / int(sizeof(T));
    static constexpr int NW = ND == 3 ? 10 : 8;          // warps
    static constexpr int WX = ND == 3 ? 1 : 8;           // x segments
    static constexpr int NPK = ND == 3 ? 33 : 32;        // packs per row segment, halo pack included
    static constexpr int SEG = NPK * VEC;                // r nodes per row segment (halo pack + owned)
    static constexpr int OWN = (NPK - 1) * VEC;          // owned x nodes per segment
    static constexpr int TX = WX * OWN, TY = ND == 3 ? 8 : 1;
    static constexpr int UW = SEG + 2 * VEC;
    static constexpr int UROWS = ND == 3 ? TY + 3 : WX;
    static constexpr int URS = ND == 3 ? UW : ((UW * int(sizeof(T)) + 127) / 128 * 128) / int(sizeof(T));
    static constexpr int UBOX_BYTES = UROWS * UW * int(sizeof(T));
    static constexpr int UTILE_BYTES = (UROWS * URS * int(sizeof(T)) + 127) / 128 * 128;
    static constexpr int FROWS = ND == 3 ? TY + 1 : WX;
    static constexpr int FBOX_BYTES = FROWS * SEG * int(sizeof(T));
    static constexpr int FTILE_BYTES = (FBOX_BYTES + 127) / 128 * 128;
    static constexpr int RPLANE = FROWS * SEG;           // elements of one r plane in shared memory
    static constexpr int NST = 4, NR = 4;
};
template <class T, int ND, bool VAR>
__host__ __device__ constexpr int res_stage_bytes() {
    return ResTile<T, ND>::UTILE_BYTES + ResTile<T, ND>::FTILE_BYTES;
}
template <class T, int ND, bool VAR>
__host__ __device__ constexpr int res_smem_bytes() {
    return res_stage_bytes<T, ND, VAR>() * ResTile<T, ND>::NST +
           ResTile<T, ND>::NR * ResTile<T, ND>::RPLANE * int(sizeof(T)) + 128;
}

template <class T, int ND, bool VAR>
__global__ void __launch_bounds__(ResTile<T, ND>::NW * 32)
k_res_tma(const __grid_constant__ CUtensorMap tmu, const __grid_constant__ CUtensorMap tmf,
          Faces<T> kf, LevelGeom g, LevelGeom gcg, Coef<T> cf, T* __restrict__ r,
          T* __restrict__ gc, double* __restrict__ partial, int mchunk) {
    pdl_start();
    using TL = ResTile<T, ND>;
    constexpr int VEC = TL::VEC;
    constexpr int STAGE = res_stage_bytes<T, ND, VAR>();
    const int tid = threadIdx.x;
    // (row R, pack lane) of this thread inside the r-tile; "lane" 0 is the halo pack
    const int wrp = tid >> 5, ln = tid & 31;
    const int R = ND == 3 ? (wrp < 9 ? wrp : (ln < 9 ? ln : 0)) : wrp;
    const int lane = ND == 3 ? (wrp < 9 ? ln + 1 : 0) : ln;
    const int NM = ND == 3 ? g.nz : g.ny;
    const long long mstride = ND == 3 ? g.pp : (long long)g.px;
    const int x0 = blockIdx.x * TL::TX;
    const int y0 = ND == 3 ? blockIdx.y * TL::TY : 0;
    const int chunk = ND == 3 ? blockIdx.z : blockIdx.y;
    const int ms = 1 + chunk * mchunk;
    const int me = min(ms + mchunk, NM - 1);
    const int nblk = gridDim.x * gridDim.y * gridDim.z;
    const int bid = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
    (void)nblk;
    if (ms >= me) { if (tid == 0) partial[bid] = 0.0; return; }
    const int mlast = (gc != nullptr && me <= NM - 2) ? me : me - 1;   // last plane computed
    const int count = mlast - ms + 3;                                  // u planes ms-1 .. mlast+1

    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);   // keeps the shared address space
    __shared__ uint64_t bars[TL::NST];
    auto us = [&](int st) { return reinterpret_cast<T*>(smem + st * STAGE); };
    auto fs = [&](int st) { return reinterpret_cast<T*>(smem + st * STAGE + TL::UTILE_BYTES); };
    T* rring = reinterpret_cast<T*>(smem + TL::NST * STAGE);

    if (tid == 0) {
        for (int s = 0; s < TL::NST; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int i) {
        const int st = i & (TL::NST - 1), p = ms - 1 + i;
        const bool wantf = i >= 1 && i <= count - 2;
        mbar_arrive_expect_tx(&bars[st], TL::UBOX_BYTES + (wantf ? TL::FBOX_BYTES : 0));
        if (ND == 3) {
            tma_load_3d(us(st), &tmu, &bars[st], x0 - 2 * VEC, y0 - 2, p);
            if (wantf) tma_load_3d(fs(st), &tmf, &bars[st], x0 - VEC, y0 - 1, p);
        } else {
            for (int w = 0; w < TL::WX; ++w) {
                tma_load_2d(us(st) + w * TL::URS, &tmu, &bars[st], x0 + w * TL::OWN - 2 * VEC, p);
                if (wantf) tma_load_2d(fs(st) + w * TL::SEG, &tmf, &bars[st], x0 + w * TL::OWN - VEC, p);
            }
        }
    };

    const int xs = ND == 3 ? x0 : x0 + R * TL::OWN;      // first owned x of this warp's segment
    const int x = xs - VEC + lane * VEC;
    const int y = ND == 3 ? y0 - 1 + R : 0;
    const int urow = ND == 3 ? R + 1 : R;
    const int voff = urow * TL::URS + VEC + lane * VEC;
    const int foff = R * TL::SEG + lane * VEC;
    const bool row_int = ND == 2 || (y > 0 && y < g.ny - 1);
    const bool owned = lane >= 1 && x < g.nx && (ND == 2 || (R >= 1 && y < g.ny));
    bool xin[VEC];
#pragma unroll
    for (int j = 0; j < VEC; ++j) xin[j] = row_int && (x + j > 0) && (x + j < g.nx - 1);

    if (tid == 0)
        for (int i = 0; i < TL::NST && i < count; ++i) issue(i);

    Pack<T> prv, cur, nxt;
    mbar_wait(&bars[0], 0);
    prv = *reinterpret_cast<const Pack<T>*>(us(0) + voff);
    mbar_wait(&bars[1], 0);
    cur = *reinterpret_cast<const Pack<T>*>(us(1) + voff);
    __syncthreads();
    if (tid == 0 && TL::NST < count) issue(TL::NST);

    double sq = 0.0;
    long long c = (long long)ms * mstride + (ND == 3 ? (long long)y * g.px : 0) + x;
    // VAR: face coefficients straight from global memory (see k_relax_tma)
    const bool kok = VAR && x >= 0 && x < g.nx && row_int;
    Pack<T> fzm, nfz, nfym, nfyp, nfx;
    T nfxl = T(0);
    auto fetch_faces = [&](const long long cc) {
        nfz = *reinterpret_cast<const Pack<T>*>(kf.z + cc);
        nfym = *reinterpret_cast<const Pack<T>*>(kf.y + cc - g.px);
        nfyp = *reinterpret_cast<const Pack<T>*>(kf.y + cc);
        nfx = *reinterpret_cast<const Pack<T>*>(kf.x + cc);
        if (x > 0) nfxl = kf.x[cc - 1];
    };
    if (kok) {
        fzm = *reinterpret_cast<const Pack<T>*>(kf.z + c - mstride);
        fetch_faces(c);
    }
    auto step = [&](auto KC, const int i) {
        constexpr int K = decltype(KC)::value;
        const int z = ms - 1 + i;
        constexpr int sn = (K + 2) & (TL::NST - 1), sc = (K + 1) & (TL::NST - 1);
        // faces of this plane were fetched one step ago; those of the next plane (it exists: z+1 <= NM-1) now
        const Pack<T> fzp = nfz, fym = nfym, fyp = nfyp, fxp = nfx;
        const T fxl = nfxl;
        if (kok) fetch_faces(c + mstride);
        mbar_wait(&bars[sn], ((i + 1) / TL::NST) & 1);
        nxt = *reinterpret_cast<const Pack<T>*>(us(sn) + voff);
        const T* vt = us(sc);
        Pack<T> dn, up;
        if (ND == 3) {
            dn = *reinterpret_cast<const Pack<T>*>(vt + voff - TL::URS);
            up = *reinterpret_cast<const Pack<T>*>(vt + voff + TL::URS);
        }
        const T vl = vt[voff - 1], vr = vt[voff + VEC];
        const Pack<T> fv = *reinterpret_cast<const Pack<T>*>(fs(sc) + foff);
        Pack<T> out;
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
            const T vc = cur.v[j];
            const T xm = j == 0 ? vl : cur.v[j - 1 < 0 ? 0 : j - 1];
            const T xp = j == VEC - 1 ? vr : cur.v[j + 1 > VEC - 1 ? VEC - 1 : j + 1];
            T Av;
            if (!VAR) {
                T s = prv.v[j] + nxt.v[j];
                if (ND == 3) s += dn.v[j] + up.v[j];
                s += xm + xp;
                Av = (cf.twod * vc - s) * cf.ih2;
            } else {
                const T fxm = j == 0 ? fxl : fxp.v[j - 1 < 0 ? 0 : j - 1];
                T acc = T(0);
                acc += fzm.v[j] * (vc - prv.v[j]);
                acc += fzp.v[j] * (vc - nxt.v[j]);
                if (ND == 3) {
                    acc += fym.v[j] * (vc - dn.v[j]);
                    acc += fyp.v[j] * (vc - up.v[j]);
                }
                acc += fxm * (vc - xm);
                acc += fxp.v[j] * (vc - xp);
                Av = acc * cf.ih2;
            }
            out.v[j] = xin[j] ? fv.v[j] - Av : T(0);
        }
        *reinterpret_cast<Pack<T>*>(rring + ((K + 1) & (TL::NR - 1)) * TL::RPLANE + foff) = out;
        if (owned && z < me) {
            if (r) *reinterpret_cast<Pack<T>*>(r + c) = out;
#pragma unroll
            for (int j = 0; j < VEC; ++j) { const double rv = double(out.v[j]); sq = __fma_rn(rv, rv, sq); }
        }
        __syncthreads();
        if (tid == 0 && i + TL::NST < count) issue(i + TL::NST);
        prv = cur; cur = nxt;
        if (VAR) fzm = fzp;
        c += mstride;
        if ((K & 1) == 0 && gc != nullptr && i >= 3) {
            // coarse plane Z = (z-1)/2 from r planes z-2, z-1, z (ring slots i-2, i-1, i)
            const int Z = (z - 1) >> 1;
            constexpr int CPR = TL::OWN / 2;                       // coarse nodes per row segment
            constexpr int NCO = CPR * (ND == 3 ? TL::TY / 2 : TL::WX);
            for (int n = tid; n < NCO; n += TL::NW * 32) {
                const int q = n / CPR, Xl = n - q * CPR;
                int X, Y, R0;
                if (ND == 3) { X = (x0 >> 1) + Xl; Y = (y0 >> 1) + q; R0 = 2 * q + 1; }
                else { X = ((x0 + q * TL::OWN) >> 1) + Xl; Y = Z; R0 = q; }
                const bool cin = X >= 1 && X <= gcg.nx - 2 && (ND == 2 || (Y >= 1 && Y <= gcg.ny - 2));
                if (!cin) continue;
                const int e0 = 2 * Xl + VEC;
                // weights are powers of two, so fma(w, r, acc) == acc + w*r bit for bit (the product is exact)
                T acc = T(0);
#pragma unroll
                for (int dm = -1; dm <= 1; ++dm) {
                    const T* rp = rring + ((K + dm) & (TL::NR - 1)) * TL::RPLANE;
#pragma unroll
                    for (int dy = (ND == 3 ? -1 : 0); dy <= (ND == 3 ? 1 : 0); ++dy) {
                        const T* rr = rp + (R0 + dy) * TL::SEG + e0;           // e0 is even: 2 scalars are one aligned load
                        const T rm = rr[-1];
                        const HalfPack<T> rc = *reinterpret_cast<const HalfPack<T>*>(rr);
                        const int m0 = (dm != 0) + (dy != 0);
                        acc = fma_rn(T(1.0 / double(1 << (ND + m0 + 1))), rm, acc);
                        acc = fma_rn(T(1.0 / double(1 << (ND + m0))), rc.v[0], acc);
                        acc = fma_rn(T(1.0 / double(1 << (ND + m0 + 1))), rc.v[1], acc);
                    }
                }
                gc[ND == 3 ? lidx(gcg, X, Y, Z) : lidx(gcg, X, Z, 0)] = acc;
            }
        }
    };
    for (int i = 1; i <= count - 2; i += 4) {
        step(std::integral_constant<int, 0>{}, i);
        if (i + 1 > count - 2) break;
        step(std::integral_constant<int, 1>{}, i + 1);
        if (i + 2 > count - 2) break;
        step(std::integral_constant<int, 2>{}, i + 2);
        if (i + 3 > count - 2) break;
        step(std::integral_constant<int, 3>{}, i + 3);
    }
    const double t = block_sum(sq);
    if (tid == 0) partial[bid] = t;
}

}  // namespace homg
