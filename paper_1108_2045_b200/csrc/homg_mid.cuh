// homg_mid.cuh — K_mid: one whole MFMG visit of a MID-size level in one launch.
//
// Levels between the K_coarse threshold (<= 9^3 / 28^2, one CTA) and the TMA-tiled threshold
// (>= 65^3 / 449^2, K_visit) neither fill the machine nor fit one CTA: their eta damped-Jacobi
// sweeps (Eq. 2-3) used to be eta launches of k_relax whose
// cost is the launch-to-launch latency, not the work (cfg2: 16 of the 32 launches of a cycle).
// Here a CTA owns a small block of nodes, loads it with a halo of `eta` nodes per side into shared
// memory (v^0 and g), and runs all eta sweeps there: sweep s is valid on the tile shrunk by s
// nodes per side, so after eta sweeps exactly the owned block is valid.  The redundant halo work
// (up to 8x in 3-D) is free on levels that cannot occupy the SMs anyway; the launch count of a
// visit drops from eta to 1.
//
// Epilogues are those of k_relax (homg_kernels.cuh): S3e bookkeeping a (+)= (d0 + v^{eta-1}) - v^0
// on the last sweep, S4 u += v^eta, and the last three iterates are stored (o0 = v^eta,
// o1 = v^{eta-1}, o2 = v^{eta-2}) because the next visit's carried variation reads them (S3c).
// None of o0/o1/o2 may alias vin (other CTAs read its halo).  Every node evaluates the expression
// trees of homg_kernels.cuh (R14): bit-identical to eta launches of k_relax.
#pragma once
#include "homg_kernels.cuh"

namespace homg {

template <class T, int ND>
struct MidTile {
    static constexpr int TX = ND == 3 ? 16 : 32, TY = ND == 3 ? 16 : 32, TZ = ND == 3 ? 16 : 1;
    static constexpr int LX = ND == 3 ? 4 : 5, LY = ND == 3 ? 4 : 5;     // log2(TX), log2(TY)
    static constexpr int N = TX * TY * TZ;
    static constexpr int NT = ND == 3 ? 512 : 256;
    static constexpr int PER = N / NT;                                    // tile nodes per thread
    static constexpr int SMEM = 3 * N * int(sizeof(T));
    static constexpr int MAX_ETA = 4;
    static_assert(N % NT == 0, "whole nodes per thread");
};

// grid = (ceil(nx / OW), ceil(ny / OW), ND == 3 ? ceil(nz / OW) : 1), OW = T - 2 eta
template <class T, int ND, bool VAR>
__global__ void __launch_bounds__(MidTile<T, ND>::NT)
k_visit_mid(LevelGeom g, Coef<T> cf, const T* __restrict__ vin, const T* __restrict__ gsrc, Faces<T> kf, int eta,
            T* __restrict__ o0, T* __restrict__ o1, T* __restrict__ o2, T* __restrict__ a, int a_assign,
            const T* __restrict__ d0, const T* __restrict__ v0, T* __restrict__ u) {
    pdl_start();
    using TL = MidTile<T, ND>;
    extern __shared__ uint4 mid_smem[];
    T* bufA = reinterpret_cast<T*>(mid_smem);
    T* bufB = bufA + TL::N;
    T* gs = bufB + TL::N;
    const int H = eta;
    const int ox = blockIdx.x * (TL::TX - 2 * H) - H, oy = blockIdx.y * (TL::TY - 2 * H) - H;
    const int oz = ND == 3 ? blockIdx.z * (TL::TZ - 2 * H) - H : 0;

    // this thread's tile nodes: n = tid + k NT  (x fastest: coalesced rows)
    long long c[TL::PER];
    unsigned char inner[TL::PER], indom[TL::PER];
#pragma unroll
    for (int k = 0; k < TL::PER; ++k) {
        const int n = threadIdx.x + k * TL::NT;
        const int lx = n & (TL::TX - 1), ly = (n >> TL::LX) & (TL::TY - 1), lz = n >> (TL::LX + TL::LY);
        const int x = ox + lx, y = oy + ly, z = oz + lz;
        const bool in = x >= 0 && x < g.nx && y >= 0 && y < g.ny && (ND == 2 || (z >= 0 && z < g.nz));
        indom[k] = in;
        inner[k] = in && is_interior<ND>(g, x, y, z);
        c[k] = lidx(g, x, y, z);
        bufA[n] = in ? vin[c[k]] : T(0);
        gs[n] = inner[k] ? gsrc[c[k]] : T(0);
    }
    // the global operands of the epilogue (S3e: d0, v^0, a; S4: u) of this thread's owned nodes are fetched
    // now, before the sweeps, so that their latency hides behind the shared-memory work
    const int OW = TL::TX - 2 * H;
    const int nown = OW * OW * (ND == 3 ? OW : 1);
    constexpr int EP = 4;                                         // eta >= 2: at most 4 owned nodes per thread
    int en[EP];
    long long ec[EP];
    bool eok[EP], ein[EP];
    T ed0[EP], ev0[EP], ea[EP], eu[EP];
#pragma unroll
    for (int i = 0; i < EP; ++i) {
        const int j = threadIdx.x + i * TL::NT;
        const int jx = j % OW, jt = j / OW, jy = jt % OW, jz = jt / OW;
        const int x = ox + H + jx, y = oy + H + jy, z = ND == 3 ? oz + H + jz : 0;
        eok[i] = j < nown && x < g.nx && y < g.ny && (ND == 2 || z < g.nz);
        ein[i] = eok[i] && is_interior<ND>(g, x, y, z);
        en[i] = ((ND == 3 ? H + jz : 0) * TL::TY + H + jy) * TL::TX + H + jx;
        ec[i] = lidx(g, x, y, z);
        ed0[i] = ev0[i] = ea[i] = eu[i] = T(0);
        if (ein[i]) {
            if (a) {
                if (d0) ed0[i] = d0[ec[i]];
                ev0[i] = v0[ec[i]];
                if (!a_assign) ea[i] = a[ec[i]];
            }
            if (u) eu[i] = u[ec[i]];
        }
    }
    __syncthreads();

    constexpr int SY = TL::TX, SZ = TL::TX * TL::TY;
    for (int it = 0; it < eta; ++it) {
        const T* vi = (it & 1) ? bufB : bufA;
        T* vo = (it & 1) ? bufA : bufB;
        const int lo = it + 1;
        T* keep2 = it == eta - 3 ? o2 : nullptr;                  // v^{eta-2} leaves shared memory two sweeps later
#pragma unroll
        for (int k = 0; k < TL::PER; ++k) {
            const int n = threadIdx.x + k * TL::NT;
            const int lx = n & (TL::TX - 1), ly = (n >> TL::LX) & (TL::TY - 1), lz = n >> (TL::LX + TL::LY);
            // the region sweep `it` is valid on
            if (lx < lo || lx >= TL::TX - lo || ly < lo || ly >= TL::TY - lo) continue;
            if (ND == 3 && (lz < lo || lz >= TL::TZ - lo)) continue;
            T vn = T(0);
            if (inner[k]) {
                const T vc = vi[n];
                if (!VAR) {
                    T s = T(0);
                    if (ND == 3) s += vi[n - SZ] + vi[n + SZ];
                    s += vi[n - SY] + vi[n + SY];
                    s += vi[n - 1] + vi[n + 1];
                    vn = jacobi_eq3(vc, s, gs[n], cf);
                } else {
                    T acc = T(0), dsum = T(0);
                    const int st[3] = {SZ, SY, 1};
                    const long long off[3] = {g.pp, (long long)g.px, 1};
                    const T* fa[3] = {kf.z, kf.y, kf.x};
#pragma unroll
                    for (int ax = 3 - ND; ax < 3; ++ax) {
                        const T fm = fa[ax][c[k] - off[ax]], fp = fa[ax][c[k]];
                        acc += fm * (vc - vi[n - st[ax]]); dsum += fm;
                        acc += fp * (vc - vi[n + st[ax]]); dsum += fp;
                    }
                    const T Av = acc * cf.ih2, D = dsum * cf.ih2;
                    vn = vc + cf.w * (gs[n] - Av) / D;
                }
            }
            vo[n] = vn;
            if (keep2 && indom[k] && lx >= H && lx < TL::TX - H && ly >= H && ly < TL::TY - H &&
                (ND == 2 || (lz >= H && lz < TL::TZ - H)))
                keep2[c[k]] = vn;
        }
        __syncthreads();
    }

    // ---- epilogue over the owned block: v^eta, v^{eta-1} out; S3e; S4 ----
    const T* vl = (eta & 1) ? bufB : bufA;                        // v^eta
    const T* vp = (eta & 1) ? bufA : bufB;                        // v^{eta-1}
#pragma unroll
    for (int i = 0; i < EP; ++i) {
        if (!eok[i]) continue;
        const T vn = vl[en[i]], vc = vp[en[i]];                   // boundary nodes hold 0
        if (o0) o0[ec[i]] = vn;
        if (o1) o1[ec[i]] = vc;
        if (!ein[i]) {
            if (a && a_assign) a[ec[i]] = T(0);
            continue;
        }
        if (a) {
            const T Dq = (ed0[i] + vc) - ev0[i];
            a[ec[i]] = a_assign ? Dq : ea[i] + Dq;
        }
        if (u) u[ec[i]] = eu[i] + vn;
    }
}

}  // namespace homg
