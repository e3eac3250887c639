// homg_literal.cuh — the paper's own design as a measured prior-art row: Algorithm L,
// the LITERAL whole-grid HOMG iteration on ONE fine-grid array (every
// iteration at every level is one launch over the whole fine grid, 1 work unit).
//
// One iteration at level m, l = 2^m, for every fine node p:
//   p on the level-m lattice (all indices multiples of l), interior:  relax with the stride-l stencil
//       (Eq. 3: neighbours p +- l e_a, h_l = l h, right-hand side g_m(p / l));
//   p on the lattice, boundary: 0;
//   every other p:  nxt(p) = cur(p) + multilinear interpolation, over the enclosing level-m cell, of the
//       lattice nodes' variation in the PREVIOUS iteration, cur - prev (one-iteration delay, L113).
// Reads only cur / prev, writes nxt.  Arithmetic and term order = oracle iteration_L (bit-identical).
#pragma once
#include "homg_kernels.cuh"

namespace homg {

// g0: the fine grid; gm: level m (g_m and, VAR, its face arrays are level-m arrays); sh = m
template <class T, int ND, bool VAR>
__global__ void k_iter_literal(LevelGeom g0, LevelGeom gm, int sh, Coef<T> cf, const T* __restrict__ cur,
                               const T* __restrict__ prev, T* __restrict__ nxt, const T* __restrict__ gsrc,
                               Faces<T> kf) {
    pdl_start();
    HOMG_NODE_XYZ(g0);
    const int l = 1 << sh, mask = l - 1;
    const long long c = lidx(g0, x, y, z);
    const bool lattice = !(x & mask) && !(y & mask) && (ND == 2 || !(z & mask));
    if (lattice) {
        if (!is_interior<ND>(g0, x, y, z)) { nxt[c] = T(0); return; }
        const long long st[3] = {g0.pp * l, (long long)g0.px * l, (long long)l};
        const long long P = lidx(gm, x >> sh, y >> sh, ND == 3 ? (z >> sh) : 0);
        const T vc = cur[c];
        if (!VAR) {
            T s = T(0);
#pragma unroll
            for (int a = 3 - ND; a < 3; ++a) s += cur[c - st[a]] + cur[c + st[a]];
            nxt[c] = jacobi_eq3(vc, s, gsrc[P], cf);
        } else {
            const long long pst[3] = {gm.pp, (long long)gm.px, 1};
            const T* fa[3] = {kf.z, kf.y, kf.x};
            T acc = T(0), ds = T(0);
#pragma unroll
            for (int a = 3 - ND; a < 3; ++a) {
                const T fm = fa[a][P - pst[a]], fp = fa[a][P];
                acc += fm * (vc - cur[c - st[a]]); ds += fm;
                acc += fp * (vc - cur[c + st[a]]); ds += fp;
            }
            const T Av = acc * cf.ih2, D = ds * cf.ih2;
            nxt[c] = vc + cf.w * (gsrc[P] - Av) / D;
        }
        return;
    }
    // multilinear weights t/l and 1 - t/l per axis (exact dyadic numbers)
    const int p[3] = {ND == 3 ? z : 0, y, x};
    const long long fst[3] = {g0.pp, (long long)g0.px, 1};
    long long base = 0;
    T wl[3] = {T(1), T(1), T(1)}, wh[3] = {T(0), T(0), T(0)};
#pragma unroll
    for (int a = 3 - ND; a < 3; ++a) {
        const int t = p[a] & mask;
        base += (long long)(p[a] - t) * fst[a];
        wh[a] = T(double(t) / double(l));
        wl[a] = T(1) - wh[a];
    }
    T acc = T(0);
#pragma unroll
    for (int c0 = 0; c0 <= (ND == 3 ? 1 : 0); ++c0)
#pragma unroll
        for (int c1 = 0; c1 <= 1; ++c1)
#pragma unroll
            for (int c2 = 0; c2 <= 1; ++c2) {
                const int cc[3] = {c0, c1, c2};
                T w = T(1);
                bool zero = false;
                long long q = base;
#pragma unroll
                for (int a = 3 - ND; a < 3; ++a) {
                    const T wa = cc[a] ? wh[a] : wl[a];
                    if (wa == T(0)) zero = true;
                    w *= wa;
                    q += (long long)cc[a] * l * fst[a];
                }
                if (zero) continue;
                acc += w * (cur[q] - prev[q]);
            }
    nxt[c] = cur[c] + acc;
}

// u += e on a whole padded array; n16 = 16-byte packs
template <class T>
__global__ void k_add_v(T* __restrict__ u, const T* __restrict__ e, long long n16) {
    pdl_start();
    constexpr int VEC = 16 / int(sizeof(T));
    struct alignas(16) P4 { T v[VEC]; };
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n16) return;
    P4 a = reinterpret_cast<const P4*>(u)[i];
    const P4 b = reinterpret_cast<const P4*>(e)[i];
#pragma unroll
    for (int j = 0; j < VEC; ++j) a.v[j] += b.v[j];
    reinterpret_cast<P4*>(u)[i] = a;
}

}  // namespace homg
