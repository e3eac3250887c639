// homg_pow2.cuh — PAPER.md section 3 (L77-85), "Power of two size grids": the whole-grid HOMG iteration on a 2-D grid
// of N = 2^k nodes per side (N-1 intervals: not nestable).  Reading: DESIGN.md R19 (Fig. 2 is not in the file).
//
//   * four subdomains of N/2 x N/2 nodes; per axis a node is in the LOW half (index < N/2) or the HIGH half;
//   * the level-m coarse points of a subdomain are marked relative to its external corner (L83): per axis
//     {i l} (low) and {N-1 - i l} (high), l = 2^m, i = 0 .. N/(2l); the last one lies just outside the subdomain —
//     the central points without which the zero mode cannot be resolved (L85);
//   * marked interior nodes relax (Eq. 3, stride l in the fine array, out-of-grid neighbours = the Dirichlet 0) with
//     the source restricted on THEIR lattice: each anchor combination is a nested lattice of the (N+1)-node grid with
//     one ghost row / column of zeros beyond the side opposite to the anchor (nested full weighting, L73);
//   * every other node adds the bilinear interpolation of the previous-iteration variations of the marked nodes of
//     its OWN subdomain's lattice (L85: no cross-domain data).
// One launch per iteration over the whole fine grid, as the paper's design has it (L51, L119).  Arithmetic and term
// order = the oracle's iteration_P / p2_restrict_all (results agree bit for bit).
#pragma once
#include "homg_kernels.cuh"

namespace homg {

template <class T>
struct P2Src {                 // the restricted source of one level on the four anchored lattices [ay * 2 + ax]
    const T* p[4];
};
template <class T>
struct P2Dst {
    T* p[4];
};

// nested full weighting on the four anchored lattices; blockIdx.z = anchor (ay * 2 + ax).
// first != 0: the fine array is the residual r itself (level 0, N x N, geometry gf), read with the anchor's flips,
// index N = the ghost (0); otherwise the fine arrays are the anchored arrays of the level below (geometry gf).
template <class T>
__global__ void k_p2_restrict(LevelGeom gc, LevelGeom gf, int N, int first, const T* __restrict__ r, P2Src<T> fine,
                              P2Dst<T> coarse) {
    pdl_start();
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int an = blockIdx.z, ay = an >> 1, ax = an & 1;
    if (x >= gc.nx || y >= gc.ny) return;
    T* out = coarse.p[an];
    const long long cc = lidx(gc, x, y, 0);
    if (x == 0 || y == 0 || x == gc.nx - 1 || y == gc.ny - 1) { out[cc] = T(0); return; }
    const T* in = first ? r : fine.p[an];
    T acc = T(0);
#pragma unroll
    for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
        for (int dx = -1; dx <= 1; ++dx) {
            const int m1 = (dy != 0) + (dx != 0);
            const T wgt = T(1.0 / double(1 << (2 + m1)));
            const int i = 2 * y + dy, j = 2 * x + dx;            // indices from the anchor
            T v;
            if (first) v = (i < N && j < N) ? in[lidx(gf, ax ? N - 1 - j : j, ay ? N - 1 - i : i, 0)] : T(0);
            else v = in[lidx(gf, j, i, 0)];
            acc += wgt * v;
        }
    out[cc] = acc;
}

// one whole-grid iteration at level sh (l = 2^sh).  src: the four anchored source arrays of that level (geometry gm);
// sh == 0: every node relaxes with the residual r itself.
template <class T>
__global__ void k_iter_p2(LevelGeom g0, LevelGeom gm, int N, int sh, Coef<T> cf, const T* __restrict__ cur,
                          const T* __restrict__ prev, T* __restrict__ nxt, const T* __restrict__ r, P2Src<T> src) {
    pdl_start();
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    if (x >= N || y >= N) return;
    const int l = 1 << sh, mask = l - 1, half = N >> 1;
    const long long c = lidx(g0, x, y, 0);
    if (x == 0 || y == 0 || x == N - 1 || y == N - 1) { nxt[c] = T(0); return; }
    // marked?  anchor 0 (low) / 1 (high) per axis
    const int tyh = N - 1 - y, txh = N - 1 - x;
    const bool ylo = !(y & mask) && y <= half, yhi = !(tyh & mask) && tyh <= half;
    const bool xlo = !(x & mask) && x <= half, xhi = !(txh & mask) && txh <= half;
    if ((ylo || yhi) && (xlo || xhi)) {
        T g;
        if (sh == 0) g = r[c];
        else {
            const int ay = ylo ? 0 : 1, ax = xlo ? 0 : 1;
            g = src.p[ay * 2 + ax][lidx(gm, (ax ? txh : x) >> sh, (ay ? tyh : y) >> sh, 0)];
        }
        auto at = [&](int yy, int xx) -> T { return (yy < 0 || yy >= N || xx < 0 || xx >= N) ? T(0) : cur[lidx(g0, xx, yy, 0)]; };
        T s = T(0);
        s += at(y - l, x) + at(y + l, x);
        s += at(y, x - l) + at(y, x + l);
        nxt[c] = jacobi_eq3(cur[c], s, g, cf);
        return;
    }
    // interpolation on the lattice of the node's own subdomain
    const int pp[2] = {y, x};
    int c0[2], c1[2];
    T wl[2], wh[2];
#pragma unroll
    for (int a = 0; a < 2; ++a) {
        const bool high = pp[a] >= half;
        const int t = high ? N - 1 - pp[a] : pp[a];
        const int i0 = t >> sh;
        wh[a] = T(double(t - (i0 << sh)) / double(l));
        wl[a] = T(1) - wh[a];
        c0[a] = high ? N - 1 - (i0 << sh) : (i0 << sh);
        c1[a] = high ? N - 1 - ((i0 + 1) << sh) : ((i0 + 1) << sh);
    }
    T acc = T(0);
#pragma unroll
    for (int cy = 0; cy < 2; ++cy)
#pragma unroll
        for (int cx = 0; cx < 2; ++cx) {
            const T wy = cy ? wh[0] : wl[0], wx = cx ? wh[1] : wl[1];
            if (wy == T(0) || wx == T(0)) continue;
            const long long q = lidx(g0, cx ? c1[1] : c0[1], cy ? c1[0] : c0[0], 0);
            acc += (wy * wx) * (cur[q] - prev[q]);
        }
    nxt[c] = cur[c] + acc;
}

}  // namespace homg
