// homg_bricks.cuh — brick forms of the level-change kernels of homg_moves.cuh (S3a deliver, S3c carried variation,
// the V cycle's prolongation).
//
// The one-pack-per-thread forms are bound by the issue rate of their scalar coarse loads: each fine pack gathers up
// to 4 coarse rows x 3 values per array, ~30 LDG.32 per 16 bytes stored (profiles/r02a: k_arrive_v takes 83 us for
// 235 MB on the 257^3 level of cfg4).  Here a thread owns the 2 x 2 fine rows (y = 2Y, 2Y+1; z = 2Z, 2Z+1) of one
// pack column: the 2 x 2 coarse rows they interpolate from are loaded ONCE (an 8-byte and a 4-byte load per row in
// fp32) and serve all four packs — 4-5 x fewer load instructions per byte moved.
// Same arithmetic, node by node and term by term, as pack_interp / deliver_pack / d0_down_pack (bit-identical).
#pragma once
#include "homg_moves.cuh"

namespace homg {

template <class T, int ND>
struct CoarseBrick {
    static constexpr int VEC = 16 / int(sizeof(T));
    static constexpr int NCV = VEC / 2 + 1;
    T c[2][2][NCV];                                  // [cz][cy][x]: (A - B) of the coarse rows (by + cy, bz + cz)
    // hy / hz: the fine rows 2Y+1 / planes 2Z+1 exist (then so do the coarse rows by+1 / bz+1)
    __device__ __forceinline__ void load(const LevelGeom& gc, const T* __restrict__ A, const T* __restrict__ B, int bx,
                                         int by, int bz, bool hy, bool hz) {
#pragma unroll
        for (int cz = 0; cz <= (ND == 3 ? 1 : 0); ++cz)
#pragma unroll
            for (int cy = 0; cy <= 1; ++cy) {
                if ((cz && !hz) || (cy && !hy)) continue;
                const long long q = lidx(gc, bx, by + cy, bz + cz);
                if (VEC == 4) {                      // bx is even: two values are one aligned 8-byte load
                    const HalfPack<T> h = *reinterpret_cast<const HalfPack<T>*>(A + q);
                    c[cz][cy][0] = h.v[0]; c[cz][cy][1] = h.v[1]; c[cz][cy][NCV - 1] = A[q + NCV - 1];
                    if (B) {
                        const HalfPack<T> g = *reinterpret_cast<const HalfPack<T>*>(B + q);
                        c[cz][cy][0] -= g.v[0]; c[cz][cy][1] -= g.v[1]; c[cz][cy][NCV - 1] -= B[q + NCV - 1];
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < NCV; ++i) {
                        c[cz][cy][i] = A[q + i];
                        if (B) c[cz][cy][i] -= B[q + i];
                    }
                }
            }
    }
    // the pack of the fine row with offsets (oy, oz) inside the brick: pack_interp's sum, term by term
    __device__ __forceinline__ Pack<T> interp(int oy, int oz) const {
        T wr = T(1);
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
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    if (j & 1) {
                        acc.v[j] += (wr * T(0.5)) * c[cz][cy][j >> 1];
                        acc.v[j] += (wr * T(0.5)) * c[cz][cy][(j >> 1) + 1];
                    } else {
                        acc.v[j] += wr * c[cz][cy][j >> 1];
                    }
                }
            }
        }
        return acc;
    }
};

#define HOMG_BRICK_XYZ(g)                                                      \
    constexpr int VEC = 16 / int(sizeof(T));                                    \
    const int x = (blockIdx.x * blockDim.x + threadIdx.x) * VEC;                \
    const int Y = blockIdx.y * blockDim.y + threadIdx.y;                        \
    const int Z = blockIdx.z;                                                   \
    if (x >= (g).nx || 2 * Y >= (g).ny || 2 * Z >= (g).nz) return;               \
    const bool hy = 2 * Y + 1 < (g).ny, hz = ND == 3 && 2 * Z + 1 < (g).nz;

template <class T, int ND>
inline dim3 grdb(const LevelGeom& g) {           // one 2 x 2 brick of pack rows per thread
    const int w = 32 * (16 / int(sizeof(T)));
    return dim3((g.nx + w - 1) / w, ((g.ny + 1) / 2 + 7) / 8, (g.nz + 1) / 2);
}

// deliver (S3a) for the four fine rows of a brick
template <class T, int ND>
__device__ __forceinline__ void deliver_brick(const LevelGeom& gf, const LevelGeom& gc, const T* __restrict__ ec,
                                              const T* __restrict__ ac, T* __restrict__ ef, T* __restrict__ af,
                                              int ef_assign, int af_mode, int x, int Y, int Z, bool hy, bool hz) {
    constexpr int VEC = 16 / int(sizeof(T));
    CoarseBrick<T, ND> br;
    if (ac) br.load(gc, ac, nullptr, x >> 1, Y, Z, hy, hz);
    const long long qc = lidx(gc, x >> 1, Y, Z);
#pragma unroll
    for (int oz = 0; oz <= (ND == 3 ? 1 : 0); ++oz)
#pragma unroll
        for (int oy = 0; oy <= 1; ++oy) {
            if ((oz && !hz) || (oy && !hy)) continue;
            const long long c = lidx(gf, x, 2 * Y + oy, 2 * Z + oz);
            Pack<T> inc;
            if (ac) inc = br.interp(oy, oz);
            else {
#pragma unroll
                for (int j = 0; j < VEC; ++j) inc.v[j] = T(0);
            }
            const bool rowcoin = !oy && !oz;
            Pack<T> e;
            if (!ef_assign) e = *reinterpret_cast<const Pack<T>*>(ef + c);
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
}

// one prolongation step of the carried variation (S3c) for the four fine rows of a brick
template <class T, int ND>
__device__ __forceinline__ void d0_down_brick(const LevelGeom& gf, const LevelGeom& gc, const T* __restrict__ A,
                                              const T* __restrict__ B, T* __restrict__ out, int coin_s, int sh,
                                              const LevelGeom& gv, const T* __restrict__ X, const T* __restrict__ Yv,
                                              int x, int Y, int Z, bool hy, bool hz) {
    constexpr int VEC = 16 / int(sizeof(T));
    CoarseBrick<T, ND> br;
    br.load(gc, A, B, x >> 1, Y, Z, hy, hz);
    const int mask = coin_s - 1;
#pragma unroll
    for (int oz = 0; oz <= (ND == 3 ? 1 : 0); ++oz)
#pragma unroll
        for (int oy = 0; oy <= 1; ++oy) {
            if ((oz && !hz) || (oy && !hy)) continue;
            const int y = 2 * Y + oy, z = 2 * Z + oz;
            Pack<T> val = br.interp(oy, oz);
            const bool rowcoin = coin_s > 0 && !(y & mask) && (ND == 2 || !(z & mask));
#pragma unroll
            for (int j = 0; j < VEC; ++j) {
                if (x + j >= gf.nx) { val.v[j] = T(0); continue; }
                if (rowcoin && !((x + j) & mask)) {
                    const long long q = lidx(gv, (x + j) >> sh, y >> sh, ND == 3 ? (z >> sh) : 0);
                    val.v[j] = X[q] - Yv[q];
                }
            }
            *reinterpret_cast<Pack<T>*>(out + lidx(gf, x, y, z)) = val;
        }
}

template <class T, int ND>
__global__ void __launch_bounds__(256)
k_deliver_b(LevelGeom gf, LevelGeom gc, const T* __restrict__ ec, const T* __restrict__ ac, T* __restrict__ ef,
            T* __restrict__ af, int ef_assign, int af_mode) {
    pdl_start();
    HOMG_BRICK_XYZ(gf);
    deliver_brick<T, ND>(gf, gc, ec, ac, ef, af, ef_assign, af_mode, x, Y, Z, hy, hz);
}

template <class T, int ND>
__global__ void __launch_bounds__(256)
k_d0_down_b(LevelGeom gf, LevelGeom gc, const T* __restrict__ A, const T* __restrict__ B, T* __restrict__ out,
            int coin_s, int sh, LevelGeom gv, const T* __restrict__ X, const T* __restrict__ Yv) {
    pdl_start();
    HOMG_BRICK_XYZ(gf);
    d0_down_brick<T, ND>(gf, gc, A, B, out, coin_s, sh, gv, X, Yv, x, Y, Z, hy, hz);
}

// one hop level m -> m-1 on the way down to a visit: deliver + the prolongation step of the carried variation
template <class T, int ND>
__global__ void __launch_bounds__(256)
k_arrive_b(LevelGeom gf, LevelGeom gc, const T* __restrict__ ec, const T* __restrict__ ac, T* __restrict__ ef,
           T* __restrict__ af, int ef_assign, int af_mode, const T* __restrict__ A, const T* __restrict__ B,
           T* __restrict__ out, int coin_s, int sh, LevelGeom gv, const T* __restrict__ X, const T* __restrict__ Yv) {
    pdl_start();
    HOMG_BRICK_XYZ(gf);
    deliver_brick<T, ND>(gf, gc, ec, ac, ef, af, ef_assign, af_mode, x, Y, Z, hy, hz);
    d0_down_brick<T, ND>(gf, gc, A, B, out, coin_s, sh, gv, X, Yv, x, Y, Z, hy, hz);
}

// Classic V-cycle, step (d): v += S^ e_c, brick form
template <class T, int ND>
__global__ void __launch_bounds__(256)
k_prolong_add_b(LevelGeom gf, LevelGeom gc, const T* __restrict__ ec, T* __restrict__ v) {
    pdl_start();
    HOMG_BRICK_XYZ(gf);
    CoarseBrick<T, ND> br;
    br.load(gc, ec, nullptr, x >> 1, Y, Z, hy, hz);
#pragma unroll
    for (int oz = 0; oz <= (ND == 3 ? 1 : 0); ++oz)
#pragma unroll
        for (int oy = 0; oy <= 1; ++oy) {
            if ((oz && !hz) || (oy && !hy)) continue;
            const long long c = lidx(gf, x, 2 * Y + oy, 2 * Z + oz);
            const Pack<T> inc = br.interp(oy, oz);
            Pack<T> vv = *reinterpret_cast<const Pack<T>*>(v + c);
#pragma unroll
            for (int j = 0; j < VEC; ++j) vv.v[j] = x + j < gf.nx ? vv.v[j] + inc.v[j] : T(0);
            *reinterpret_cast<Pack<T>*>(v + c) = vv;
        }
}

}  // namespace homg
