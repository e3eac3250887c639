// homg_kernels.cuh — generic per-level CUDA kernels of the HOMG cycle (sm_100a).
//
// These are the "any level, any schedule" kernels: one thread per node, coalesced along x.
// The level-0 / large-level fast paths (register blocking along the slowest axis, TMA tile
// staging, fused interpolate+correct+relax, fused residual+restriction) live in
// homg_fused.cuh; the persistent coarse-level kernel in homg_coarse.cuh.  All of them
// compute the same expressions, defined here in node_* device functions.
//
// Layout of one level array: nodes INCLUDING the Dirichlet
// boundary, index = z*pp + y*px + x, px = row pitch (multiple of 128 B), pp = px*ny.
// Boundary entries and pad columns are 0 and are never written with anything else.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "homg_geom.h"

namespace homg {

// Programmatic dependent launch: let the next kernel of the stream begin its launch now, then wait
// until every kernel before this one has completed and flushed its writes.  Must precede the first
// global access of a kernel; a no-op when the launch carries no programmatic attribute.
__device__ __forceinline__ void pdl_start() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

__device__ __forceinline__ long long lidx(const LevelGeom& g, int x, int y, int z) {
    return (long long)z * g.pp + (long long)y * g.px + x;
}

template <int ND>
__device__ __forceinline__ bool is_interior(const LevelGeom& g, int x, int y, int z) {
    bool in = x > 0 && x < g.nx - 1 && y > 0 && y < g.ny - 1;
    if (ND == 3) in = in && z > 0 && z < g.nz - 1;
    return in;
}

// harmonic-mean face coefficient between two nodal values (R11)
template <class T>
__device__ __forceinline__ T kface(T kc, T kq) { return T(2) * kc * kq / (kc + kq); }

// (A v)(c) and the diagonal D(c) at one interior node.  Constant coefficient:
// (2d v - sum_nb v)/h^2, D = 2d/h^2.  Variable: sum_faces kf (v_c - v_q)/h^2, D = sum kf/h^2.
// Neighbour order: slowest axis first (z, y, x), minus then plus (Eq.3).
template <class T, int ND, bool VAR>
__device__ __forceinline__ void node_A(const T* __restrict__ v, const Faces<T>& kf, long long c,
                                       const LevelGeom& g, const Coef<T>& cf, T& Av, T& D) {
    if (!VAR) {
        T s = T(0);
        if (ND == 3) s += v[c - g.pp] + v[c + g.pp];
        s += v[c - g.px] + v[c + g.px];
        s += v[c - 1] + v[c + 1];
        Av = (cf.twod * v[c] - s) * cf.ih2;
        D = cf.twod * cf.ih2;
    } else {
        const T vc = v[c];
        T acc = T(0), dsum = T(0);
        const long long off[3] = {g.pp, (long long)g.px, 1};
        const T* fa[3] = {kf.z, kf.y, kf.x};
#pragma unroll
        for (int a = 3 - ND; a < 3; ++a) {
            const T fm = fa[a][c - off[a]], fp = fa[a][c];       // faces towards the - and + neighbour
            acc += fm * (vc - v[c - off[a]]); dsum += fm;
            acc += fp * (vc - v[c + off[a]]); dsum += fp;
        }
        Av = acc * cf.ih2;
        D = dsum * cf.ih2;
    }
}

__device__ __forceinline__ float fma_rn(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double fma_rn(double a, double b, double c) { return __fma_rn(a, b, c); }

// constant-coefficient damped Jacobi, Eq. 3 in the sign convention of DESIGN.md R1:
//   v + w_p ((sum_nb v - 2d v) + h_l^2 g),  w_p = w / 2d;  s = the neighbour sum (slowest axis first).
// The three multiply-adds are single fused operations, in the same places as the oracle's std::fma
// calls (R14), so every kernel that sweeps agrees with it bit for bit.
template <class T>
__device__ __forceinline__ T jacobi_eq3(T vc, T s, T gval, const Coef<T>& cf) {
    T t = fma_rn(-cf.twod, vc, s);
    t = fma_rn(cf.h2, gval, t);
    return fma_rn(cf.wp, t, vc);
}

// damped Jacobi at one interior node
template <class T, int ND, bool VAR>
__device__ __forceinline__ T node_jacobi(const T* __restrict__ v, const Faces<T>& k, T gval,
                                         long long c, const LevelGeom& g, const Coef<T>& cf) {
    if (!VAR) {
        T s = T(0);
        if (ND == 3) s += v[c - g.pp] + v[c + g.pp];
        s += v[c - g.px] + v[c + g.px];
        s += v[c - 1] + v[c + 1];
        return jacobi_eq3(v[c], s, gval, cf);
    }
    T Av, D;
    node_A<T, ND, VAR>(v, k, c, g, cf, Av, D);
    return v[c] + cf.w * (gval - Av) / D;
}

// ---------------------------------------------------------------------------------------
// thread -> node mapping of the generic kernels: blockDim = (32, 8, 1), grid covers
// (nx, ny, nz) of the OUTPUT level.
// ---------------------------------------------------------------------------------------
#define HOMG_NODE_XYZ(g)                                        \
    int x = blockIdx.x * blockDim.x + threadIdx.x;              \
    int y = blockIdx.y * blockDim.y + threadIdx.y;              \
    int z = blockIdx.z;                                         \
    if (x >= (g).nx || y >= (g).ny || z >= (g).nz) return;

// block-wide sum in double: warp shuffles, then one value per warp through shared memory.
// Returns the total in thread 0 of the block.
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double wsum[32];
    int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    int nthr = blockDim.x * blockDim.y * blockDim.z;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((tid & 31) == 0) wsum[tid >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (tid < 32) {
        t = tid < (nthr + 31) / 32 ? wsum[tid] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    __syncthreads();
    return t;
}

// r = f - A u on interior nodes, 0 on the boundary; per-block partial of sum r^2 (double)
// -> partial[linear block id].  r may be null (norm only).
template <class T, int ND, bool VAR>
__global__ void k_residual(LevelGeom g, Coef<T> cf, const T* __restrict__ u, const T* __restrict__ f,
                           Faces<T> k, T* __restrict__ r, double* __restrict__ partial) {
    pdl_start();
    int x = blockIdx.x * blockDim.x + threadIdx.x;
    int y = blockIdx.y * blockDim.y + threadIdx.y;
    int z = blockIdx.z;
    double sq = 0.0;
    if (x < g.nx && y < g.ny && z < g.nz) {
        long long c = lidx(g, x, y, z);
        T rv = T(0);
        if (is_interior<ND>(g, x, y, z)) {
            T Av, D;
            node_A<T, ND, VAR>(u, k, c, g, cf, Av, D);
            rv = f[c] - Av;
        }
        if (r) r[c] = rv;
        sq = double(rv) * double(rv);
    }
    double t = block_sum(sq);
    if (threadIdx.x == 0 && threadIdx.y == 0)
        partial[blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = t;
}

// fixed-order sum of the per-block partials -> hist[*slot]; optionally ++*slot.
// One block of 256 threads.  The order is fixed, so norms are reproducible run to run.
__global__ void k_norm_finish(const double* __restrict__ partial, int n, double* __restrict__ hist,
                              int* __restrict__ slot, int cap, int advance, double* __restrict__ scalar_out) {
    pdl_start();
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) s += partial[i];
    double t = block_sum(s);
    if (threadIdx.x == 0) {
        if (scalar_out) *scalar_out = t;
        if (hist) {
            int c = *slot;
            if (c < cap) hist[c] = t;
            if (advance) *slot = c + 1;
        }
    }
}

// homg_solve: the same sum; the new norm^2 goes to hist[*slot] and decides whether the device-side loop (a CUDA
// graph WHILE node) runs another cycle: while ||r_c||^2 > tol^2 ||r_0||^2 and c < max_cycles   (PAPER.md L75:
// "restart the cycles as many times as needed to reach any desired accuracy")
struct SolveParams {
    double tol2;        // (relative tolerance)^2
    int max_slot;       // history index at which the loop stops regardless (cycles already issued + max_cycles)
};
__global__ void k_norm_finish_solve(const double* __restrict__ partial, int n, double* __restrict__ hist,
                                    int* __restrict__ slot, int cap, const SolveParams* __restrict__ sp,
                                    unsigned long long cond) {
    pdl_start();
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) s += partial[i];
    double t = block_sum(s);
    if (threadIdx.x == 0) {
        const int c = *slot;
        if (c < cap) hist[c] = t;
        *slot = c + 1;
        const double first = c == 0 ? t : hist[0];
        const bool go = c < sp->max_slot && c + 1 < cap && t > sp->tol2 * first;
        cudaGraphSetConditional(cudaGraphConditionalHandle(cond), go ? 1u : 0u);
    }
}

// full weighting: coarse interior node I = sum_{delta in {-1,0,1}^d} 2^(-d-|delta|_1) fine(2I+delta);
// coarse boundary entries 0.  Grid over the COARSE level.
template <class T, int ND>
__global__ void k_restrict(LevelGeom gc, LevelGeom gf, const T* __restrict__ fine, T* __restrict__ coarse) {
    pdl_start();
    HOMG_NODE_XYZ(gc);
    long long cc = lidx(gc, x, y, z);
    if (!is_interior<ND>(gc, x, y, z)) { coarse[cc] = T(0); return; }
    long long fc = lidx(gf, 2 * x, 2 * y, ND == 3 ? 2 * z : 0);
    T acc = T(0);
#pragma unroll
    for (int dz = (ND == 3 ? -1 : 0); dz <= (ND == 3 ? 1 : 0); ++dz)
#pragma unroll
        for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
            for (int dx = -1; dx <= 1; ++dx) {
                int m1 = (dz != 0) + (dy != 0) + (dx != 0);
                T wgt = T(1.0 / double(1 << (ND + m1)));
                acc += wgt * fine[fc + dz * gf.pp + dy * (long long)gf.px + dx];
            }
    coarse[cc] = acc;
}

// multilinear interpolation of coarse array(s) at fine node (x,y,z): sum over the corners of
// the enclosing coarse cell of prod_a (1/2 | 1 | 0) * (A[q] - B[q])  (B nullable).
template <class T, int ND>
__device__ __forceinline__ T node_interp(const LevelGeom& gc, const T* __restrict__ A, const T* __restrict__ B,
                                         int x, int y, int z) {
    int bx = x >> 1, by = y >> 1, bz = ND == 3 ? (z >> 1) : 0;
    int ox = x & 1, oy = y & 1, oz = ND == 3 ? (z & 1) : 0;
    T acc = T(0);
#pragma unroll
    for (int cz = 0; cz <= (ND == 3 ? 1 : 0); ++cz)
#pragma unroll
        for (int cy = 0; cy <= 1; ++cy)
#pragma unroll
            for (int cx = 0; cx <= 1; ++cx) {
                // weight per axis: odd offset -> 1/2 for both corners; even -> 1 for corner 0, 0 for corner 1
                if ((cx && !ox) || (cy && !oy) || (cz && !oz)) continue;
                T w = T(1);
                if (ox) w *= T(0.5);
                if (oy) w *= T(0.5);
                if (ND == 3 && oz) w *= T(0.5);
                long long q = lidx(gc, bx + cx, by + cy, bz + cz);
                T val = A[q];
                if (B) val -= B[q];
                acc += w * val;
            }
    return acc;
}

// deliver level m -> m-1 (S3a): inc = S^ a_c; coincident nodes take
// e_c, the others add inc; if af != null (fine level >= 1) af += inc.  Grid over the FINE level.
// ac == null means a_c = 0 (nothing pending).  ef_assign: e_f is known to be 0 (first time this
// level is reached in the cycle) so the sum is an assignment; af_mode 0: none, 1: af += inc,
// 2: af = inc (a_f known to be 0).  These flags only remove memsets / reads of known zeros.
template <class T, int ND>
__global__ void k_deliver(LevelGeom gf, LevelGeom gc, const T* __restrict__ ec, const T* __restrict__ ac,
                          T* __restrict__ ef, T* __restrict__ af, int ef_assign, int af_mode) {
    pdl_start();
    HOMG_NODE_XYZ(gf);
    long long c = lidx(gf, x, y, z);
    T inc = ac ? node_interp<T, ND>(gc, ac, nullptr, x, y, z) : T(0);
    bool coin = !(x & 1) && !(y & 1) && (ND == 2 || !(z & 1));
    if (coin) ef[c] = ec[lidx(gc, x >> 1, y >> 1, ND == 3 ? (z >> 1) : 0)];
    else ef[c] = ef_assign ? inc : ef[c] + inc;
    if (af_mode == 1) af[c] += inc;
    else if (af_mode == 2) af[c] = inc;
}

// inject level m-1 -> m: e_c(P) = e_f(2P).  Grid over the COARSE level.   (one array)
template <class T, int ND>
__global__ void k_inject(LevelGeom gc, LevelGeom gf, const T* __restrict__ ef, T* __restrict__ ec) {
    pdl_start();
    HOMG_NODE_XYZ(gc);
    ec[lidx(gc, x, y, z)] = ef[lidx(gf, 2 * x, 2 * y, ND == 3 ? 2 * z : 0)];
}

// carried variation when the target level t is the same or coarser than the last visited level v:
// d0(P) = (X - Y)(P * s)  with dl = X - Y on level v.  Grid over level t.     (S3c)
template <class T, int ND>
__global__ void k_d0_up(LevelGeom gt, LevelGeom gv, int s, const T* __restrict__ X, const T* __restrict__ Y,
                        T* __restrict__ d0) {
    pdl_start();
    HOMG_NODE_XYZ(gt);
    long long q = lidx(gv, x * s, y * s, ND == 3 ? z * s : 0);
    d0[lidx(gt, x, y, z)] = X[q] - Y[q];
}

// a move up that ends on level t: the last inject (level t-1 -> t) and k_d0_up have the same grid and
// independent outputs — one launch instead of two
template <class T, int ND>
__global__ void k_rise(LevelGeom gt, LevelGeom gf, const T* __restrict__ ef, T* __restrict__ ec, LevelGeom gv, int s,
                       const T* __restrict__ X, const T* __restrict__ Y, T* __restrict__ d0) {
    pdl_start();
    HOMG_NODE_XYZ(gt);
    const long long c = lidx(gt, x, y, z);
    ec[c] = ef[lidx(gf, 2 * x, 2 * y, ND == 3 ? 2 * z : 0)];
    const long long q = lidx(gv, x * s, y * s, ND == 3 ? z * s : 0);
    d0[c] = X[q] - Y[q];
}

// one prolongation step of the carried variation going finer: out = S^(A - B) on the fine level;
// on the last step (coin_s > 0) nodes coincident with level v (all indices multiples of coin_s)
// take dl = X - Y of level v instead.  Grid over the FINE level.               (S3c)
template <class T, int ND>
__global__ void k_d0_down(LevelGeom gf, LevelGeom gc, const T* __restrict__ A, const T* __restrict__ B,
                          T* __restrict__ out, int coin_s, LevelGeom gv, const T* __restrict__ X,
                          const T* __restrict__ Y) {
    pdl_start();
    HOMG_NODE_XYZ(gf);
    T val;
    bool coin = coin_s > 0 && (x % coin_s == 0) && (y % coin_s == 0) && (ND == 2 || (z % coin_s == 0));
    if (coin) {
        long long q = lidx(gv, x / coin_s, y / coin_s, ND == 3 ? z / coin_s : 0);
        val = X[q] - Y[q];
    } else {
        val = node_interp<T, ND>(gc, A, B, x, y, z);
    }
    out[lidx(gf, x, y, z)] = val;
}

// one damped-Jacobi sweep on a level (S3d), with the optional fused epilogues:
//   a != null : a += (d0 + vin) - v0          (S3e; on the sweep whose INPUT is v^{eta-1})
//   u != null : u += vout                      (S4;  on the last sweep of the cycle)
//   d0 == null means d0 = 0 (first visit of a cycle); a_assign: a is known to be 0.
// Boundary nodes are written too (with 0) so a buffer that held an older iterate is fully defined.
template <class T, int ND, bool VAR>
__global__ void k_relax(LevelGeom g, Coef<T> cf, const T* __restrict__ vin, const T* __restrict__ gsrc,
                        Faces<T> k, T* __restrict__ vout, T* __restrict__ a, int a_assign,
                        const T* __restrict__ d0, const T* __restrict__ v0, T* __restrict__ u) {
    pdl_start();
    HOMG_NODE_XYZ(g);
    long long c = lidx(g, x, y, z);
    if (!is_interior<ND>(g, x, y, z)) {
        vout[c] = T(0);
        if (a && a_assign) a[c] = T(0);
        return;
    }
    T vn = node_jacobi<T, ND, VAR>(vin, k, gsrc[c], c, g, cf);
    vout[c] = vn;
    if (a) {
        T D = ((d0 ? d0[c] : T(0)) + vin[c]) - v0[c];
        a[c] = a_assign ? D : a[c] + D;
    }
    if (u) u[c] += vn;
}

// dense user array (C order, nx contiguous) <-> padded level-0 array.  to_padded: boundary -> 0.
template <class T, int ND>
__global__ void k_pack(LevelGeom g, const T* __restrict__ dense, T* __restrict__ padded, int zero_boundary) {
    pdl_start();
    HOMG_NODE_XYZ(g);
    long long d = ((long long)z * g.ny + y) * g.nx + x;
    T v = dense[d];
    if (zero_boundary && !is_interior<ND>(g, x, y, z)) v = T(0);
    padded[lidx(g, x, y, z)] = v;
}

template <class T, int ND>
__global__ void k_unpack(LevelGeom g, const T* __restrict__ padded, T* __restrict__ dense) {
    pdl_start();
    HOMG_NODE_XYZ(g);
    dense[((long long)z * g.ny + y) * g.nx + x] = padded[lidx(g, x, y, z)];
}

// mixed-precision outer loop: padded array of one precision -> padded array of another
// (the row pitches differ), dst = TO(src) or dst += TO(src); one thread per node incl. the boundary
template <class TO, class FROM, int ND, bool ADD>
__global__ void k_cvt_pad(LevelGeom gto, LevelGeom gfrom, const FROM* __restrict__ src, TO* __restrict__ dst) {
    pdl_start();
    HOMG_NODE_XYZ(gto);
    const long long d = lidx(gto, x, y, z);
    const TO v = TO(src[lidx(gfrom, x, y, z)]);
    dst[d] = ADD ? dst[d] + v : v;
}

// the same for the two level-0 passes of every mixed cycle, four x nodes per thread (rows of both arrays
// start 128-B aligned): r32 = float(r64)  /  u64 += double(e32)
template <int ND, bool ADD>
__global__ void __launch_bounds__(256)
k_cvt4(LevelGeom g64, LevelGeom g32, double* __restrict__ d64, float* __restrict__ f32) {
    pdl_start();
    const int x = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g64.nx || y >= g64.ny || z >= g64.nz) return;
    double2* p64 = reinterpret_cast<double2*>(d64 + lidx(g64, x, y, z));
    float4* p32 = reinterpret_cast<float4*>(f32 + lidx(g32, x, y, z));
    if (ADD) {
        const float4 e = *p32;
        double2 a = p64[0], b = p64[1];
        a.x += double(e.x); a.y += double(e.y); b.x += double(e.z); b.y += double(e.w);
        p64[0] = a; p64[1] = b;
    } else {
        const double2 a = p64[0], b = p64[1];
        *p32 = make_float4(float(a.x), float(a.y), float(b.x), float(b.y));
    }
}

// S0: face coefficients of one level from its nodal k (R11); 0 where the + neighbour does not exist
template <class T, int ND>
__global__ void k_faces(LevelGeom g, const T* __restrict__ k, T* __restrict__ fz, T* __restrict__ fy, T* __restrict__ fx) {
    pdl_start();
    HOMG_NODE_XYZ(g);
    const long long c = lidx(g, x, y, z);
    const T kc = k[c];
    fx[c] = x + 1 < g.nx ? kface(kc, k[c + 1]) : T(0);
    fy[c] = y + 1 < g.ny ? kface(kc, k[c + g.px]) : T(0);
    if (ND == 3) fz[c] = z + 1 < g.nz ? kface(kc, k[c + g.pp]) : T(0);
}

// S0: wd = omega / D at every interior node, D = (sum of the 2d face coefficients) / h^2 summed in the sweep's own order
// (z-, z+, y-, y+, x-, x+), so that D is the very number the sweeps compute; 0 on the boundary.  Read by the
// variable-coefficient form of K_visit, which then needs neither the sum nor the division per sweep (R14).
template <class T, int ND>
__global__ void k_wdiag(LevelGeom g, Coef<T> cf, Faces<T> kf, T* __restrict__ wd) {
    pdl_start();
    HOMG_NODE_XYZ(g);
    const long long c = lidx(g, x, y, z);
    if (!is_interior<ND>(g, x, y, z)) { wd[c] = T(0); return; }
    T ds = T(0);
    if (ND == 3) { ds += kf.z[c - g.pp]; ds += kf.z[c]; }
    ds += kf.y[c - g.px]; ds += kf.y[c];
    ds += kf.x[c - 1]; ds += kf.x[c];
    wd[c] = cf.w / (ds * cf.ih2);
}

// coefficient sampling onto the next level: k_c(P) = k_f(2P)     (R11)
// (same kernel as k_inject; kept under its own name for the profile listing)
template <class T, int ND>
__global__ void k_sample_coef(LevelGeom gc, LevelGeom gf, const T* __restrict__ kf, T* __restrict__ kc) {
    pdl_start();
    HOMG_NODE_XYZ(gc);
    kc[lidx(gc, x, y, z)] = kf[lidx(gf, 2 * x, 2 * y, ND == 3 ? 2 * z : 0)];
}

}  // namespace homg
