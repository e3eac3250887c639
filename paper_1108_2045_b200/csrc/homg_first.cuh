// homg_first.cuh — K_relax, first sweep of a visit: interpolate + correct + relax in ONE pass
// (north_star item 2; "interpolation and relaxation are the same task", L113).
//
// When the MFMG schedule arrives on a large level f from the next coarser level c, the correction on
// f before the first Jacobi sweep is (Algorithm H, S3a, first arrival in the cycle):
//       v0(p) = e_c(p/2)                       p coincident with a level-c node
//       v0(p) = (S^ a_c)(p)                    otherwise (multilinear interpolation of the pending
//                                              increments of level c)
// This kernel never writes v0: a CTA stages the coarse planes of e_c and a_c by TMA, builds the fine
// plane of v0 (tile + halo) in shared memory, and runs the Jacobi sweep of homg_fused.cuh on it,
// writing only v1.  HBM traffic: read g_f, write v1, read two coarse arrays = (2 + 2/2^d) passes
// instead of (1 + 2/2^d) + 3 for deliver-then-sweep.
//
// Geometry: as K_res — a warp row holds 32 packs, pack 0 is recomputed halo (x0-VEC..x0-1), packs
// 1..31 are owned, plus one scalar halo node on the right; 3-D: 10 warps = rows y0-1..y0+8 of the
// fine tile, of which warps 1..8 relax; 2-D: 8 warps = 8 x-segments of one row.
#pragma once
#include "homg_fused.cuh"

namespace homg {

template <class T, int ND>
struct FirstTile {
    static constexpr int ES = int(sizeof(T));
    static constexpr int VEC = 16 / ES;
    static constexpr int NW = ND == 3 ? 10 : 8;
    static constexpr int WX = ND == 3 ? 1 : 8;
    static constexpr int SEG = 32 * VEC, OWN = 31 * VEC;
    static constexpr int TX = WX * OWN, TY = ND == 3 ? 8 : 1;
    // fine tile rows (also the k tile): 33 packs wide; 2-D rows are TMA destinations -> 128-B stride
    static constexpr int FW = 33 * VEC;
    static constexpr int FROWS = ND == 3 ? TY + 2 : WX;
    static constexpr int FRS = ND == 3 ? FW : ((FW * ES + 127) / 128 * 128) / ES;
    static constexpr int FPLANE = FROWS * FRS;                       // elements
    static constexpr int NF = 4;                                     // fine ring slots
    // coarse tiles of e_c and a_c
    // TMA needs the box to START on a 16-B boundary of the row: the box begins at the coarse column
    // (xs-VEC)/2 rounded down to a multiple of VEC, so it is up to VEC/2 columns wider than needed.
    static constexpr int CW = ((16 * VEC + 1 + VEC / 2) * ES + 15) / 16 * 16 / ES;
    static constexpr int CROWS = ND == 3 ? TY / 2 + 2 : WX;
    static constexpr int CRS = ND == 3 ? CW : ((CW * ES + 127) / 128 * 128) / ES;
    static constexpr int CBOX_BYTES = CROWS * CW * ES;
    static constexpr int CTILE_BYTES = (CROWS * CRS * ES + 127) / 128 * 128;
    static constexpr int NC = 4;                                     // coarse ring slots
    // g tile
    static constexpr int GROWS = ND == 3 ? TY : WX;
    static constexpr int GBOX_BYTES = GROWS * SEG * ES;
    static constexpr int NG = 4;                                     // ring of the fine-keyed TMA stages (g, k)
};
template <class T, int ND, bool VAR>
__host__ __device__ constexpr int first_gk_stage_bytes() {
    return FirstTile<T, ND>::GBOX_BYTES;
}
template <class T, int ND, bool VAR>
__host__ __device__ constexpr int first_smem_bytes() {
    using TL = FirstTile<T, ND>;
    return TL::NG * first_gk_stage_bytes<T, ND, VAR>() + TL::NC * 2 * TL::CTILE_BYTES +
           (TL::NF * TL::FPLANE * TL::ES + 127) / 128 * 128 + 128;
}


// tme / tma_ : tensor maps of e_c and a_c (level c = f+1);  tmg : g_f;  kf : face coefficients (VAR).
// vout = v1;  u != null: u += v1 (a visit of a single sweep that ends the cycle).  mchunk even.
template <class T, int ND, bool VAR>
__global__ void __launch_bounds__(FirstTile<T, ND>::NW * 32)
k_relax_first(const __grid_constant__ CUtensorMap tme, const __grid_constant__ CUtensorMap tma_,
              const __grid_constant__ CUtensorMap tmg, Faces<T> kf, LevelGeom g,
              Coef<T> cf, T* __restrict__ vout, T* __restrict__ u, int mchunk) {
    pdl_start();
    using TL = FirstTile<T, ND>;
    constexpr int VEC = TL::VEC;
    constexpr int NCV = VEC / 2 + 1;
    constexpr int GK = first_gk_stage_bytes<T, ND, VAR>();
    const int tid = threadIdx.x, lane = tid & 31, R = tid >> 5;
    const int NM = ND == 3 ? g.nz : g.ny;
    const long long mstride = ND == 3 ? g.pp : (long long)g.px;
    const int x0 = blockIdx.x * TL::TX;
    const int y0 = ND == 3 ? blockIdx.y * TL::TY : 0;
    const int chunk = ND == 3 ? blockIdx.z : blockIdx.y;
    const int ms = 1 + chunk * mchunk;
    const int me = min(ms + mchunk, NM - 1);
    if (ms >= me) return;
    const int nq = me - ms + 2;                 // fine planes q = 0..nq-1  <->  p = ms-1+q
    const int Z0 = (ms - 1) >> 1;               // first coarse plane (ms is odd)
    const int ncz = (nq >> 1) + 1;              // coarse planes Z0 .. Z0+ncz-1

    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    __shared__ uint64_t fbar[TL::NG], cbar[TL::NC];
    auto gs = [&](int st) { return reinterpret_cast<T*>(smem + st * GK); };
    unsigned char* cbase = smem + TL::NG * GK;
    auto ce = [&](int st) { return reinterpret_cast<T*>(cbase + (2 * st) * TL::CTILE_BYTES); };
    auto ca = [&](int st) { return reinterpret_cast<T*>(cbase + (2 * st + 1) * TL::CTILE_BYTES); };
    T* fring = reinterpret_cast<T*>(cbase + TL::NC * 2 * TL::CTILE_BYTES);

    if (tid == 0) {
        for (int s = 0; s < TL::NG; ++s) mbar_init(&fbar[s], 1);
        for (int s = 0; s < TL::NC; ++s) mbar_init(&cbar[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    auto issue_f = [&](int q) {                 // g and k of fine plane q
        const int st = q & (TL::NG - 1), p = ms - 1 + q;
        const bool wantg = q >= 1 && q <= nq - 2;
        const uint32_t bytes = wantg ? TL::GBOX_BYTES : 0;
        if (bytes == 0) { mbar_arrive_expect_tx(&fbar[st], 0); return; }   // keeps the phase count = q / NG
        mbar_arrive_expect_tx(&fbar[st], bytes);
        if (ND == 3) {
            if (wantg) tma_load_3d(gs(st), &tmg, &fbar[st], x0 - VEC, y0, p);
        } else {
            for (int w = 0; w < TL::WX; ++w) {
                if (wantg) tma_load_2d(gs(st) + w * TL::SEG, &tmg, &fbar[st], x0 + w * TL::OWN - VEC, p);
            }
        }
    };
    auto issue_c = [&](int zc) {                // e_c and a_c of coarse plane Z0+zc
        const int st = zc & (TL::NC - 1), Z = Z0 + zc;
        mbar_arrive_expect_tx(&cbar[st], 2 * TL::CBOX_BYTES);
        if (ND == 3) {
            const int X = (x0 - VEC) / 2;
            tma_load_3d(ce(st), &tme, &cbar[st], X - (X & (VEC - 1)), y0 / 2 - 1, Z);
            tma_load_3d(ca(st), &tma_, &cbar[st], X - (X & (VEC - 1)), y0 / 2 - 1, Z);
        } else {
            for (int w = 0; w < TL::WX; ++w) {
                const int X = (x0 + w * TL::OWN - VEC) / 2;
                tma_load_2d(ce(st) + w * TL::CRS, &tme, &cbar[st], X - (X & (VEC - 1)), Z);
                tma_load_2d(ca(st) + w * TL::CRS, &tma_, &cbar[st], X - (X & (VEC - 1)), Z);
            }
        }
    };
    if (tid == 0) {
        for (int zc = 0; zc < TL::NC && zc < ncz; ++zc) issue_c(zc);
        for (int q = 0; q < TL::NG && q < nq; ++q) issue_f(q);
    }

    // ---- this thread's place ----
    const int xs = ND == 3 ? x0 : x0 + R * TL::OWN;          // first owned x of the segment
    const int x = xs - VEC + lane * VEC;
    const int y = ND == 3 ? y0 - 1 + R : 0;
    const int foff = R * TL::FRS + lane * VEC;               // my pack in a fine / k tile
    const int goff = (ND == 3 ? R - 1 : R) * TL::SEG + lane * VEC;
    const int yl = ND == 3 ? (R + 1) >> 1 : R;               // my (lower) coarse row
    const bool yodd = ND == 3 && !(R & 1);
    const int coff = yl * TL::CRS + (((xs - VEC) / 2) & (VEC - 1)) + lane * (VEC / 2);   // + the box's alignment shift
    const bool relaxer = ND == 2 || (R >= 1 && R <= TL::TY);
    const bool row_int = ND == 2 || (y > 0 && y < g.ny - 1);
    const bool owned = relaxer && lane >= 1 && x < g.nx && (ND == 2 || y < g.ny);
    bool xin[VEC];
#pragma unroll
    for (int j = 0; j < VEC; ++j) xin[j] = row_int && (x + j > 0) && (x + j < g.nx - 1);

    // S3a in shared memory: fine plane q of v0 from the coarse planes (q>>1) and ((q+1)>>1)
    auto produce = [&](const int q) {
        const bool zodd = q & 1;
        const int zlo = q >> 1, zhi = (q + 1) >> 1;
        mbar_wait(&cbar[zlo & (TL::NC - 1)], (zlo / TL::NC) & 1);
        if (zodd) mbar_wait(&cbar[zhi & (TL::NC - 1)], (zhi / TL::NC) & 1);
        const T* A0 = ca(zlo & (TL::NC - 1)) + coff;
        const T* A1 = ca(zhi & (TL::NC - 1)) + coff;
        const T* E0 = ce(zlo & (TL::NC - 1)) + coff;
        T acc[VEC];
        T accx = T(0);
        constexpr int xoff = NCV - 1;                         // lane 31: the right halo node's coarse column
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
            accx = first ? c[NCV - 1] : accx + c[NCV - 1];
        };
        addrow(A0, true);
        if (yodd) addrow(A0 + TL::CRS, false);
        if (zodd) {
            addrow(A1, false);
            if (yodd) addrow(A1 + TL::CRS, false);
        }
        const T wzy = (zodd && yodd) ? T(0.25) : ((zodd || yodd) ? T(0.5) : T(1));
        const bool coin = !zodd && !yodd;
        Pack<T> out;
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
            if (j & 1) out.v[j] = (T(0.5) * wzy) * acc[j];
            else out.v[j] = coin ? E0[j >> 1] : wzy * acc[j];
        }
        T* ft = fring + (q & (TL::NF - 1)) * TL::FPLANE;
        *reinterpret_cast<Pack<T>*>(ft + foff) = out;
        if (lane == 31) ft[foff + VEC] = coin ? E0[xoff] : wzy * accx;
    };

    produce(0);
    if (nq > 1) produce(1);
    Pack<T> prv, cur, nxt;
    __syncthreads();
    prv = *reinterpret_cast<const Pack<T>*>(fring + foff);
    cur = *reinterpret_cast<const Pack<T>*>(fring + TL::FPLANE + foff);
    if (tid == 0 && TL::NC < ncz) issue_c(TL::NC);

    long long c = (long long)ms * mstride + (ND == 3 ? (long long)y * g.px : 0) + x;
    // VAR: face coefficients straight from global memory (see k_relax_tma)
    const bool kok = VAR && relaxer && x >= 0 && x < g.nx && row_int;
    Pack<T> fzm;
    if (kok) fzm = *reinterpret_cast<const Pack<T>*>(kf.z + c - mstride);
    auto step = [&](auto KC, const int q) {
        constexpr int K = decltype(KC)::value;              // (q-1) mod 4
        constexpr int sc = (K + 1) & 3, sn = (K + 2) & 3;    // ring slots of planes q and q+1
        produce(q + 1);
        __syncthreads();
        if (tid == 0) {
            if (q + 3 < nq) issue_f(q + 3);
            // q even (K odd): coarse plane q/2 was last used by produce(q+1) above
            if ((K & 1) && (q >> 1) + TL::NC < ncz) issue_c((q >> 1) + TL::NC);
        }
        if (relaxer) {
            Pack<T> fzp, fym, fyp, fxp;
            T fxl = T(0);
            if (kok) {
                fzp = *reinterpret_cast<const Pack<T>*>(kf.z + c);
                fym = *reinterpret_cast<const Pack<T>*>(kf.y + c - g.px);
                fyp = *reinterpret_cast<const Pack<T>*>(kf.y + c);
                fxp = *reinterpret_cast<const Pack<T>*>(kf.x + c);
                if (x > 0) fxl = kf.x[c - 1];
            }
            mbar_wait(&fbar[sc], (q / TL::NG) & 1);
            const T* vn = fring + sn * TL::FPLANE;
            const T* vt = fring + sc * TL::FPLANE;
            nxt = *reinterpret_cast<const Pack<T>*>(vn + foff);
            Pack<T> dn, up;
            if (ND == 3) {
                dn = *reinterpret_cast<const Pack<T>*>(vt + foff - TL::FRS);
                up = *reinterpret_cast<const Pack<T>*>(vt + foff + TL::FRS);
            }
            const T vl = vt[foff - 1], vr = vt[foff + VEC];
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
            if (owned) {
                if (vout) *reinterpret_cast<Pack<T>*>(vout + c) = out;
                if (u) {
                    Pack<T> uu = *reinterpret_cast<const Pack<T>*>(u + c);
#pragma unroll
                    for (int j = 0; j < VEC; ++j) uu.v[j] += out.v[j];
                    *reinterpret_cast<Pack<T>*>(u + c) = uu;
                }
            }
            prv = cur; cur = nxt;
            if (VAR) fzm = fzp;
        }
        c += mstride;
    };
    for (int q = 1; q <= nq - 2; q += 4) {
        step(std::integral_constant<int, 0>{}, q);
        if (q + 1 > nq - 2) break;
        step(std::integral_constant<int, 1>{}, q + 1);
        if (q + 2 > nq - 2) break;
        step(std::integral_constant<int, 2>{}, q + 2);
        if (q + 3 > nq - 2) break;
        step(std::integral_constant<int, 3>{}, q + 3);
    }
}

}  // namespace homg
