// homg_moves.cuh — vectorised level-change kernels for the LARGE levels: S3a deliver (interpolate +
// correct onto a pass-through level) and S3c (prolongation of the carried variation).  Same
// arithmetic, node by node and term by term, as k_deliver / k_d0_down of homg_kernels.cuh (results
// are bit-identical); a thread owns one 16-byte pack of consecutive x nodes, so the fine arrays move
// as LDG.128 / STG.128 and every coarse value is loaded once per pack instead of once per node.
//
#pragma once
#include "homg_fused.cuh"

namespace homg {

// multilinear interpolation of (A - B) (B nullable) at the VEC fine nodes x..x+VEC-1 of row (y, z);
// x is a multiple of VEC.  Term order per node = node_interp: cz outer, cy, cx inner.
template <class T, int ND>
__device__ __forceinline__ Pack<T> pack_interp(const LevelGeom& gc, const T* __restrict__ A, const T* __restrict__ B,
                                               int x, int y, int z) {
    constexpr int VEC = 16 / int(sizeof(T));
    constexpr int NCV = VEC / 2 + 1;
    const int bx = x >> 1, by = y >> 1, bz = ND == 3 ? (z >> 1) : 0;
    const int oy = y & 1, oz = ND == 3 ? (z & 1) : 0;
    T wr = T(1);                                   // weight of the row part (y, z)
    if (oy) wr *= T(0.5);
    if (oz) wr *= T(0.5);
    Pack<T> acc;
#pragma unroll
    for (int j = 0; j < VEC; ++j) acc.v[j] = T(0);
#pragma unroll
    for (int cz = 0; cz <= (ND == 3 ? 1 : 0); ++cz) {
        if (cz && !oz) continue;
#pragma unroll
        for (int cy = 0; cy <= 1; ++cy) {
            if (cy && !oy) continue;
            const long long q = lidx(gc, bx, by + cy, bz + cz);
            T c[NCV];
#pragma unroll
            for (int i = 0; i < NCV; ++i) {
                c[i] = A[q + i];
                if (B) c[i] -= B[q + i];
            }
#pragma unroll
            for (int j = 0; j < VEC; ++j) {
                if (j & 1) {
                    acc.v[j] += (wr * T(0.5)) * c[j >> 1];
                    acc.v[j] += (wr * T(0.5)) * c[(j >> 1) + 1];
                } else {
                    acc.v[j] += wr * c[j >> 1];
                }
            }
        }
    }
    return acc;
}

#define HOMG_PACK_XYZ(g)                                                       \
    constexpr int VEC = 16 / int(sizeof(T));                                    \
    const int x = (blockIdx.x * blockDim.x + threadIdx.x) * VEC;                \
    const int y = blockIdx.y * blockDim.y + threadIdx.y;                        \
    const int z = blockIdx.z;                                                   \
    if (x >= (g).nx || y >= (g).ny || z >= (g).nz) return;

// k_deliver for the pack x..x+VEC-1 of row (y, z)
template <class T, int ND>
__device__ __forceinline__ void deliver_pack(const LevelGeom& gf, const LevelGeom& gc, const T* __restrict__ ec,
                                             const T* __restrict__ ac, T* __restrict__ ef, T* __restrict__ af,
                                             int ef_assign, int af_mode, int x, int y, int z) {
    constexpr int VEC = 16 / int(sizeof(T));
    const long long c = lidx(gf, x, y, z);
    Pack<T> inc;
    if (ac) inc = pack_interp<T, ND>(gc, ac, nullptr, x, y, z);
    else {
#pragma unroll
        for (int j = 0; j < VEC; ++j) inc.v[j] = T(0);
    }
    const bool rowcoin = !(y & 1) && (ND == 2 || !(z & 1));
    Pack<T> e;
    if (!ef_assign) e = *reinterpret_cast<const Pack<T>*>(ef + c);
    const long long qc = lidx(gc, x >> 1, y >> 1, ND == 3 ? (z >> 1) : 0);
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
        if (x + j >= gf.nx) { e.v[j] = T(0); inc.v[j] = T(0); continue; }     // pad columns stay 0
        if (rowcoin && !(j & 1)) e.v[j] = ec[qc + (j >> 1)];
        else e.v[j] = ef_assign ? inc.v[j] : e.v[j] + inc.v[j];
    }
    *reinterpret_cast<Pack<T>*>(ef + c) = e;
    if (af_mode == 1) {
        Pack<T> a = *reinterpret_cast<const Pack<T>*>(af + c);
#pragma unroll
        for (int j = 0; j < VEC; ++j) a.v[j] += inc.v[j];
        *reinterpret_cast<Pack<T>*>(af + c) = a;
    } else if (af_mode == 2) {
        *reinterpret_cast<Pack<T>*>(af + c) = inc;
    }
}

// k_d0_down for one pack; coin_s is 0 or a power of two (sh = log2 coin_s)
template <class T, int ND>
__device__ __forceinline__ void d0_down_pack(const LevelGeom& gf, const LevelGeom& gc, const T* __restrict__ A,
                                             const T* __restrict__ B, T* __restrict__ out, int coin_s, int sh,
                                             const LevelGeom& gv, const T* __restrict__ X, const T* __restrict__ Y,
                                             int x, int y, int z) {
    constexpr int VEC = 16 / int(sizeof(T));
    Pack<T> val = pack_interp<T, ND>(gc, A, B, x, y, z);
    const int mask = coin_s - 1;
    const bool rowcoin = coin_s > 0 && !(y & mask) && (ND == 2 || !(z & mask));
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
        if (x + j >= gf.nx) { val.v[j] = T(0); continue; }
        if (rowcoin && !((x + j) & mask)) {
            const long long q = lidx(gv, (x + j) >> sh, y >> sh, ND == 3 ? (z >> sh) : 0);
            val.v[j] = X[q] - Y[q];
        }
    }
    *reinterpret_cast<Pack<T>*>(out + lidx(gf, x, y, z)) = val;
}

// one pack per thread.  grid = (ceil(nx / (32 VEC)), ceil(ny / 8), nz), block (32, 8).
template <class T, int ND>
__global__ void __launch_bounds__(256)
k_deliver_v(LevelGeom gf, LevelGeom gc, const T* __restrict__ ec, const T* __restrict__ ac, T* __restrict__ ef,
            T* __restrict__ af, int ef_assign, int af_mode) {
    pdl_start();
    HOMG_PACK_XYZ(gf);
    deliver_pack<T, ND>(gf, gc, ec, ac, ef, af, ef_assign, af_mode, x, y, z);
}

template <class T, int ND>
__global__ void __launch_bounds__(256)
k_d0_down_v(LevelGeom gf, LevelGeom gc, const T* __restrict__ A, const T* __restrict__ B, T* __restrict__ out,
            int coin_s, int sh, LevelGeom gv, const T* __restrict__ X, const T* __restrict__ Y) {
    pdl_start();
    HOMG_PACK_XYZ(gf);
    d0_down_pack<T, ND>(gf, gc, A, B, out, coin_s, sh, gv, X, Y, x, y, z);
}

// one hop level m -> m-1 on the way down to a visit: S3a deliver and the S3c prolongation step of the
// carried variation have the same grid and independent outputs — one launch instead of two
template <class T, int ND>
__global__ void __launch_bounds__(256)
k_arrive_v(LevelGeom gf, LevelGeom gc, const T* __restrict__ ec, const T* __restrict__ ac, T* __restrict__ ef,
           T* __restrict__ af, int ef_assign, int af_mode, const T* __restrict__ A, const T* __restrict__ B,
           T* __restrict__ out, int coin_s, int sh, LevelGeom gv, const T* __restrict__ X, const T* __restrict__ Y) {
    pdl_start();
    HOMG_PACK_XYZ(gf);
    deliver_pack<T, ND>(gf, gc, ec, ac, ef, af, ef_assign, af_mode, x, y, z);
    d0_down_pack<T, ND>(gf, gc, A, B, out, coin_s, sh, gv, X, Y, x, y, z);
}

// Classic V-cycle, step (d): v += S^ e_c on every node (coincident nodes add e_c itself,
// weight 1).  One pack per thread, fine array updated in place.
template <class T, int ND>
__global__ void __launch_bounds__(256)
k_prolong_add_v(LevelGeom gf, LevelGeom gc, const T* __restrict__ ec, T* __restrict__ v) {
    pdl_start();
    HOMG_PACK_XYZ(gf);
    const long long c = lidx(gf, x, y, z);
    const Pack<T> inc = pack_interp<T, ND>(gc, ec, nullptr, x, y, z);
    Pack<T> vv = *reinterpret_cast<const Pack<T>*>(v + c);
#pragma unroll
    for (int j = 0; j < VEC; ++j) vv.v[j] = x + j < gf.nx ? vv.v[j] + inc.v[j] : T(0);
    *reinterpret_cast<Pack<T>*>(v + c) = vv;
}

// Classic V-cycle, step (c) on a coarsest level with ONE interior node (3^d grid): the exact solve
// e = g / D, evaluated in double as the oracle's 1x1 LU does (D = the operator's diagonal in T).
template <class T, int ND, bool VAR>
__global__ void k_coarsest_solve(LevelGeom g, Coef<T> cf, const T* __restrict__ gsrc, Faces<T> kf,
                                 T* __restrict__ e) {
    pdl_start();
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const long long c = lidx(g, 1, 1, ND == 3 ? 1 : 0);
    T D;
    if (!VAR) {
        D = cf.twod * cf.ih2;
    } else {
        T acc = T(0);
        const long long off[3] = {g.pp, (long long)g.px, 1};
        const T* fa[3] = {kf.z, kf.y, kf.x};
#pragma unroll
        for (int a = 3 - ND; a < 3; ++a) {
            acc += fa[a][c - off[a]] * (T(1) - T(0));
            acc += fa[a][c] * (T(1) - T(0));
        }
        D = acc * cf.ih2;
    }
    e[c] = T(double(gsrc[c]) / double(D));
}

}  // namespace homg
