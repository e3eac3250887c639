// homg_coarse.cuh — K_coarse: the coarse-level path of the HOMG cycle (north_star item 4).
//
// The small levels of the hierarchy cannot fill the machine and are latency-bound: issuing one
// launch per whole-level operation (the occupancy problem the paper is about)
// costs more in launch gaps than in work.  Here every maximal run of consecutive operations whose
// OUTPUT level is small is ONE launch of one thread-block cluster that interprets a short program
// (CoarseOp records written by the executor into device memory once, when the cycle is first
// recorded); operations are separated by a cluster barrier instead of a kernel boundary.
//
// Every operation computes exactly the expression trees of homg_kernels.cuh (R14), so the
// result is bit-identical to the per-level launches.  Data written earlier in the same launch is
// read with ld.global.cg (L2), never through the non-coherent path.
#pragma once
#include <cooperative_groups.h>

#include "homg_kernels.cuh"

namespace homg {

enum { OP_ZERO = 0, OP_RESTRICT, OP_DELIVER, OP_INJECT, OP_D0_UP, OP_D0_DOWN, OP_RELAX, OP_RELAXN };

constexpr int kRelaxnSmemMax = 176 * 1024;   // dynamic shared memory an OP_RELAXN may ask for

template <class T>
struct CoarseOp {
    int type;
    int act;                  // 1: a tiny level, worked by CTA 0 alone; 0: by the whole cluster
    int f0, f1, s;            // flags / stride (meaning per type, as the arguments of the generic kernel)
    long long count;          // OP_ZERO: elements
    LevelGeom go, gi, gv;     // output level, input level, level of the last visit (D0_DOWN)
    Coef<T> cf;
    Faces<T> kf;              // OP_RELAX, variable coefficient
    const T* p[5];
    T* q[3];
    T* qx[2];                 // OP_RELAXN: where v^{eta-1} and v^{eta-2} go (q[0]: v^eta); null = not kept
};

constexpr int kMaxRunOps = 96;   // records staged in shared memory per launch; longer runs are split

// CG = true: ld.global.cg (L2) — required when another CTA of the cluster wrote the data earlier in
// this launch.  CG = false (single-CTA run): plain loads; the CTA barrier orders them after the CTA's
// own earlier stores (CUDA memory model), and they may hit L1.
template <bool CG, class T>
__device__ __forceinline__ T ldg_(const T* p) { return CG ? __ldcg(p) : *p; }
#define ldcg ldg_<CG>

// (A v)(c), D(c): homg_kernels.cuh node_A, with L2 loads
template <class T, int ND, bool VAR, bool CG>
__device__ __forceinline__ void cnode_A(const T* v, const Faces<T>& kf, long long c, const LevelGeom& g, const Coef<T>& cf,
                                        T vc, T& Av, T& D) {
    if (!VAR) {
        T s = T(0);
        if (ND == 3) s += ldcg(v + c - g.pp) + ldcg(v + c + g.pp);
        s += ldcg(v + c - g.px) + ldcg(v + c + g.px);
        s += ldcg(v + c - 1) + ldcg(v + c + 1);
        Av = (cf.twod * vc - s) * cf.ih2;
        D = cf.twod * cf.ih2;
    } else {
        T acc = T(0), dsum = T(0);
        const long long off[3] = {g.pp, (long long)g.px, 1};
        const T* fa[3] = {kf.z, kf.y, kf.x};                 // written once at set_coefficient: plain loads
#pragma unroll
        for (int a = 3 - ND; a < 3; ++a) {
            const T fm = fa[a][c - off[a]], fp = fa[a][c];
            acc += fm * (vc - ldcg(v + c - off[a])); dsum += fm;
            acc += fp * (vc - ldcg(v + c + off[a])); dsum += fp;
        }
        Av = acc * cf.ih2;
        D = dsum * cf.ih2;
    }
}

// homg_kernels.cuh node_interp, with L2 loads
template <class T, int ND, bool CG>
__device__ __forceinline__ T cnode_interp(const LevelGeom& gc, const T* A, const T* B, int x, int y, int z) {
    int bx = x >> 1, by = y >> 1, bz = ND == 3 ? (z >> 1) : 0;
    int ox = x & 1, oy = y & 1, oz = ND == 3 ? (z & 1) : 0;
    T acc = T(0);
#pragma unroll
    for (int cz = 0; cz <= (ND == 3 ? 1 : 0); ++cz)
#pragma unroll
        for (int cy = 0; cy <= 1; ++cy)
#pragma unroll
            for (int cx = 0; cx <= 1; ++cx) {
                if ((cx && !ox) || (cy && !oy) || (cz && !oz)) continue;
                T w = T(1);
                if (ox) w *= T(0.5);
                if (oy) w *= T(0.5);
                if (ND == 3 && oz) w *= T(0.5);
                long long q = lidx(gc, bx + cx, by + cy, bz + cz);
                T val = ldcg(A + q);
                if (B) val -= ldcg(B + q);
                acc += w * val;
            }
    return acc;
}

template <class T, int ND, bool VAR, bool CG>
__device__ __forceinline__ void coarse_node(const CoarseOp<T>& o, int x, int y, int z) {
    const LevelGeom& g = o.go;
    const long long c = lidx(g, x, y, z);
    switch (o.type) {
    case OP_RESTRICT: {                                   // k_restrict
        if (!is_interior<ND>(g, x, y, z)) { o.q[0][c] = T(0); return; }
        const LevelGeom& gf = o.gi;
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
                    acc += wgt * ldcg(o.p[0] + fc + dz * gf.pp + dy * (long long)gf.px + dx);
                }
        o.q[0][c] = acc;
        return;
    }
    case OP_DELIVER: {                                    // k_deliver: f0 = ef_assign, f1 = af_mode
        const LevelGeom& gc = o.gi;
        T inc = o.p[1] ? cnode_interp<T, ND, CG>(gc, o.p[1], nullptr, x, y, z) : T(0);
        bool coin = !(x & 1) && !(y & 1) && (ND == 2 || !(z & 1));
        T* ef = o.q[0];
        T* af = o.q[1];
        if (coin) ef[c] = ldcg(o.p[0] + lidx(gc, x >> 1, y >> 1, ND == 3 ? (z >> 1) : 0));
        else ef[c] = o.f0 ? inc : ldcg(ef + c) + inc;
        if (o.f1 == 1) af[c] = ldcg(af + c) + inc;
        else if (o.f1 == 2) af[c] = inc;
        return;
    }
    case OP_INJECT:                                       // k_inject
        o.q[0][c] = ldcg(o.p[0] + lidx(o.gi, 2 * x, 2 * y, ND == 3 ? 2 * z : 0));
        return;
    case OP_D0_UP: {                                      // k_d0_up
        long long q = lidx(o.gi, x * o.s, y * o.s, ND == 3 ? z * o.s : 0);
        o.q[0][c] = ldcg(o.p[0] + q) - ldcg(o.p[1] + q);
        return;
    }
    case OP_D0_DOWN: {                                    // k_d0_down: s = coin_s
        T val;
        const int cs = o.s;
        bool coin = cs > 0 && (x % cs == 0) && (y % cs == 0) && (ND == 2 || (z % cs == 0));
        if (coin) {
            long long q = lidx(o.gv, x / cs, y / cs, ND == 3 ? z / cs : 0);
            val = ldcg(o.p[2] + q) - ldcg(o.p[3] + q);
        } else {
            val = cnode_interp<T, ND, CG>(o.gi, o.p[0], o.p[1], x, y, z);
        }
        o.q[0][c] = val;
        return;
    }
    case OP_RELAX: {                                      // k_relax: f0 = a_assign
        T* vout = o.q[0];
        T* a = o.q[1];
        T* u = o.q[2];
        if (!is_interior<ND>(g, x, y, z)) {
            vout[c] = T(0);
            if (a && o.f0) a[c] = T(0);
            return;
        }
        const T vc = ldcg(o.p[0] + c);
        T vn;
        if (!VAR) {
            const T* v = o.p[0];
            T s = T(0);
            if (ND == 3) s += ldcg(v + c - g.pp) + ldcg(v + c + g.pp);
            s += ldcg(v + c - g.px) + ldcg(v + c + g.px);
            s += ldcg(v + c - 1) + ldcg(v + c + 1);
            vn = jacobi_eq3(vc, s, ldcg(o.p[1] + c), o.cf);
        } else {
            T Av, D;
            cnode_A<T, ND, VAR, CG>(o.p[0], o.kf, c, g, o.cf, vc, Av, D);
            vn = vc + o.cf.w * (ldcg(o.p[1] + c) - Av) / D;
        }
        vout[c] = vn;
        if (a) {
            T Dq = ((o.p[3] ? ldcg(o.p[3] + c) : T(0)) + vc) - ldcg(o.p[4] + c);
            a[c] = o.f0 ? Dq : ldcg(a + c) + Dq;
        }
        if (u) u[c] = ldcg(u + c) + vn;
        return;
    }
    default: return;
    }
}

#undef ldcg

// OP_RELAXN: ALL `o.s` = eta sweeps of a visit on a small level by one CTA, the iterate kept in shared
// memory between sweeps (compact nx*ny*nz layout: two ping-pong copies of v and one of g), one CTA
// barrier per sweep instead of one record (and one L2 round trip) per sweep.  Only the last three
// iterates are written to their global buffers (the next visit's carried variation reads them, S3c);
// the last sweep carries the epilogues of OP_RELAX.  Same arithmetic, node by node, as OP_RELAX.
template <class T, int ND, bool VAR, bool CG>
__device__ void coarse_relaxn(const CoarseOp<T>& o, T* sm) {
    const LevelGeom& g = o.go;
    const int nx = g.nx, ny = g.ny, nz = g.nz, N = nx * ny * nz, eta = o.s;
    const int sy = nx, sz = nx * ny;
    T* bufA = sm;
    T* bufB = sm + N;
    T* gs = sm + 2 * N;
    for (int n = threadIdx.x; n < N; n += blockDim.x) {
        const int x = n % nx, t = n / nx;
        const long long c = lidx(g, x, t % ny, t / ny);
        bufA[n] = ldg_<CG>(o.p[0] + c);
        gs[n] = ldg_<CG>(o.p[1] + c);
    }
    __syncthreads();
    long long c = 0;
    bool inner = false;
    for (int it = 0; it < eta; ++it) {
        const T* vin = (it & 1) ? bufB : bufA;
        T* vout = (it & 1) ? bufA : bufB;
        const bool last = it == eta - 1;
        T* gout = last ? o.q[0] : (it == eta - 2 ? o.qx[0] : (it == eta - 3 ? o.qx[1] : nullptr));
        T* a = last ? o.q[1] : nullptr;
        T* u = last ? o.q[2] : nullptr;
        for (int n = threadIdx.x; n < N; n += blockDim.x) {
            // (the integer divisions are a long dependent chain: a thread with a single node keeps its
            // coordinates from the first sweep)
            if (it == 0 || N > int(blockDim.x)) {
                const int x = n % nx, t = n / nx, y = t % ny, z = t / ny;
                c = lidx(g, x, y, z);
                inner = is_interior<ND>(g, x, y, z);
            }
            if (!inner) {
                vout[n] = T(0);
                if (gout) gout[c] = T(0);
                if (a && o.f0) a[c] = T(0);
                continue;
            }
            const T vc = vin[n];
            T vn;
            if (!VAR) {
                T s = T(0);
                if (ND == 3) s += vin[n - sz] + vin[n + sz];
                s += vin[n - sy] + vin[n + sy];
                s += vin[n - 1] + vin[n + 1];
                vn = jacobi_eq3(vc, s, gs[n], o.cf);
            } else {
                T acc = T(0), dsum = T(0);
                const int st[3] = {sz, sy, 1};
                const long long off[3] = {g.pp, (long long)g.px, 1};
                const T* fa[3] = {o.kf.z, o.kf.y, o.kf.x};
#pragma unroll
                for (int ax = 3 - ND; ax < 3; ++ax) {
                    const T fm = fa[ax][c - off[ax]], fp = fa[ax][c];
                    acc += fm * (vc - vin[n - st[ax]]); dsum += fm;
                    acc += fp * (vc - vin[n + st[ax]]); dsum += fp;
                }
                const T Av = acc * o.cf.ih2, D = dsum * o.cf.ih2;
                vn = vc + o.cf.w * (gs[n] - Av) / D;
            }
            vout[n] = vn;
            if (gout) gout[c] = vn;
            if (a) {
                const T Dq = ((o.p[3] ? ldg_<CG>(o.p[3] + c) : T(0)) + vc) - ldg_<CG>(o.p[4] + c);
                a[c] = o.f0 ? Dq : ldg_<CG>(a + c) + Dq;
            }
            if (u) u[c] = ldg_<CG>(u + c) + vn;
        }
        __syncthreads();
    }
}

// One launch = one cluster of gridDim.x CTAs x 1024 threads running ops[0..nops), nops <= kMaxRunOps.
// MULTI = (gridDim.x > 1).  Operations on tiny levels (act = 1) are worked by CTA 0 alone and
// separated by a CTA barrier; everything else by the whole cluster and a cluster barrier.
template <class T, int ND, bool VAR, bool MULTI>
__global__ void __launch_bounds__(1024) k_coarse_run(const CoarseOp<T>* __restrict__ ops, int nops) {
    pdl_start();
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    __shared__ CoarseOp<T> sops[kMaxRunOps];
    extern __shared__ uint4 relaxn_smem[];                // OP_RELAXN: 3 compact copies of a small level
    {   // the records were written by the host before the launch: plain loads are safe
        const int words = nops * int(sizeof(CoarseOp<T>) / 4);
        for (int w = threadIdx.x; w < words; w += blockDim.x)
            reinterpret_cast<unsigned*>(sops)[w] = reinterpret_cast<const unsigned*>(ops)[w];
    }
    __syncthreads();
    for (int i = 0; i < nops; ++i) {
        const CoarseOp<T>& op = sops[i];
        const bool solo = !MULTI || op.act == 1;
        if (!solo || blockIdx.x == 0) {
            const unsigned nth = solo ? blockDim.x : gridDim.x * blockDim.x;
            const unsigned gt = solo ? threadIdx.x : blockIdx.x * blockDim.x + threadIdx.x;
            if (op.type == OP_ZERO) {
                for (long long n = gt; n < op.count; n += nth) op.q[0][n] = T(0);
            } else if (op.type == OP_RELAXN) {             // act = 1: this CTA alone
                coarse_relaxn<T, ND, VAR, MULTI>(op, reinterpret_cast<T*>(relaxn_smem));
            } else {
                const int nx = op.go.nx, ny = op.go.ny;
                const int total = nx * ny * op.go.nz;
                for (int n = gt; n < total; n += nth) {
                    const int x = n % nx;
                    const int t = n / nx;
                    coarse_node<T, ND, VAR, MULTI>(op, x, t % ny, t / ny);
                }
            }
        }
        if (i + 1 == nops) break;
        if (!MULTI) __syncthreads();
        else if (op.act == 1 && sops[i + 1].act == 1) { if (blockIdx.x == 0) __syncthreads(); }
        else cluster.sync();                    // release/acquire at cluster scope: orders the global writes
    }
}

}  // namespace homg
