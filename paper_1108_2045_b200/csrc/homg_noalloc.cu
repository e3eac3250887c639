// homg_noalloc.cu — ONE entry point that allocates nothing: homg_residual_norm_noalloc (include/homg.h).
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
// forbid it) and so cannot create a homg_solver (whose residual kernel keeps its per-block partial sums in the
// caller-allocated workspace).  This is the residual-norm step S1/S5 (r = f - A u, ||r||_2) of the
// constant-coefficient stencils on DENSE device arrays, a variant of k_residual / k_norm_finish (homg_kernels.cuh)
// whose scratch —
// one fp64 partial of sum r^2 per block — lives in a file-scope static __device__ array of kNoAllocMaxBlocks
// doubles (1 MiB; every GPU that loads libhomg.so holds it until the process exits).
//
// Rules this file follows:
//   * in host code `g_noalloc_partial` is a host-side stand-in, NOT a device address: the device address is taken
//     once per device, with that device current, by cudaGetSymbolAddress (checked), and passed to the kernels;
//   * no cudaMalloc / cudaFree / allocating library routine is called;
//   * grids that need more than kNoAllocMaxBlocks partials are rejected with HOMG_EINVAL and a message;
//   * every call shares the array and finds the previous call's contents in it: every block of a launch WRITES its
//     partial (nothing is accumulated into the array, nothing must start at zero) and the finishing kernel reads
//     exactly the entries this call's grid wrote; CALLS THAT OVERLAP ON THE GPU (two streams, two threads) RACE on
//     the array — serialise them.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/homg.h"
#include "homg_geom.h"

namespace homg {
namespace noalloc {

constexpr int kNoAllocMaxBlocks = 131072;          // partials: 131072 x 8 B = 1 MiB per GPU
constexpr int kNoAllocMaxDevices = 64;

static __device__ __align__(256) double g_noalloc_partial[kNoAllocMaxBlocks];

// (homg_kernels.cuh defines non-template kernels and cannot be included from a second translation unit: the few
// device helpers this file needs are restated here — same expressions, R14)
__device__ __forceinline__ long long lidx(const LevelGeom& g, int x, int y, int z) {
    return (long long)z * g.pp + (long long)y * g.px + x;
}
template <int ND>
__device__ __forceinline__ bool is_interior(const LevelGeom& g, int x, int y, int z) {
    bool in = x > 0 && x < g.nx - 1 && y > 0 && y < g.ny - 1;
    if (ND == 3) in = in && z > 0 && z < g.nz - 1;
    return in;
}
// (A v)(c) = (2d v - sum_nb v) / h^2, neighbours summed slowest axis first, minus then plus
template <class T, int ND>
__device__ __forceinline__ T node_A_const(const T* __restrict__ v, long long c, const LevelGeom& g, T twod, T ih2) {
    T s = T(0);
    if (ND == 3) s += v[c - g.pp] + v[c + g.pp];
    s += v[c - g.px] + v[c + g.px];
    s += v[c - 1] + v[c + 1];
    return (twod * v[c] - s) * ih2;
}
// block-wide sum in double: warp shuffles, then one value per warp through shared memory; total in thread 0
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double wsum[32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthr = blockDim.x * blockDim.y * blockDim.z;
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

// r = f - A u on the interior nodes of a dense array (px = nx, pp = nx ny), sum r^2 per block -> partial[block]
// (the variant of k_residual: same node_A, same block_sum; r itself is not stored)
template <class T, int ND>
__global__ void __launch_bounds__(256)
k_residual_norm_dense(LevelGeom g, T twod, T ih2, const T* __restrict__ u, const T* __restrict__ f, double* __restrict__ partial) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    double sq = 0.0;
    if (x < g.nx && y < g.ny && z < g.nz && is_interior<ND>(g, x, y, z)) {
        const long long c = lidx(g, x, y, z);
        const T rv = f[c] - node_A_const<T, ND>(u, c, g, twod, ih2);
        sq = double(rv) * double(rv);
    }
    const double t = block_sum(sq);
    if (threadIdx.x == 0 && threadIdx.y == 0)
        partial[blockIdx.x + gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z)] = t;   // written, never accumulated
}

// fixed-order sum of the n partials this call wrote -> *out = sqrt(sum)   (one block of 256 threads)
__global__ void k_norm_finish_dense(const double* __restrict__ partial, int n, double* __restrict__ out) {
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) s += partial[i];
    const double t = block_sum(s);
    if (threadIdx.x == 0) *out = sqrt(t);
}

namespace {

std::mutex g_mu;
double* g_partial_dev[kNoAllocMaxDevices] = {};    // device address of g_noalloc_partial, per device

// set-up, once per device, with that device current
cudaError_t scratch_address(double** out, int* dev_out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *dev_out = dev;
    if (dev < 0 || dev >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_partial_dev[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_noalloc_partial);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_partial_dev[dev] = p;
    }
    *out = g_partial_dev[dev];
    return cudaSuccess;
}

homg_status fail(homg_status st, char* err, size_t cap, const char* msg) {
    if (err && cap) std::snprintf(err, cap, "%s", msg);
    return st;
}

template <class T, int ND>
cudaError_t run(const LevelGeom& g, double h, const void* u, const void* f, double* partial, int nblocks, dim3 grid,
                double* out, cudaStream_t st) {
    k_residual_norm_dense<T, ND><<<grid, dim3(32, 8, 1), 0, st>>>(g, T(2 * ND), T(1.0 / (h * h)), static_cast<const T*>(u),
                                                                   static_cast<const T*>(f), partial);
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) return e;
    k_norm_finish_dense<<<1, 256, 0, st>>>(partial, nblocks, out);
    return cudaPeekAtLastError();
}

}  // namespace
}  // namespace noalloc
}  // namespace homg

using namespace homg;
using namespace homg::noalloc;

extern "C" homg_status homg_residual_norm_noalloc(int ndim, const int64_t* dims, homg_dtype dtype, double h, const void* u_dev,
                                                  const void* f_dev, double* norm_out_dev, void* cuda_stream, char* err,
                                                  size_t err_cap) {
    if (err && err_cap) err[0] = 0;
    if (!dims || !u_dev || !f_dev || !norm_out_dev) return fail(HOMG_EINVAL, err, err_cap, "homg_residual_norm_noalloc: null pointer");
    if (ndim != 2 && ndim != 3) return fail(HOMG_EINVAL, err, err_cap, "homg_residual_norm_noalloc: ndim must be 2 or 3");
    if (dtype != HOMG_F32 && dtype != HOMG_F64) return fail(HOMG_EINVAL, err, err_cap, "homg_residual_norm_noalloc: dtype must be HOMG_F32 or HOMG_F64");
    for (int a = 0; a < ndim; ++a)
        if (dims[a] < 3 || dims[a] > (int64_t(1) << 20)) return fail(HOMG_EINVAL, err, err_cap, "homg_residual_norm_noalloc: dims out of range");
    LevelGeom g;
    g.nz = ndim == 3 ? int(dims[0]) : 1;
    g.ny = int(dims[ndim - 2]);
    g.nx = int(dims[ndim - 1]);
    g.px = g.nx;
    g.pp = (long long)g.nx * g.ny;
    if (!(h > 0)) h = 1.0 / double(dims[0] - 1);
    const long long gx = (g.nx + 31) / 32, gy = (g.ny + 7) / 8, gz = g.nz;
    const long long nblocks = gx * gy * gz;
    if (nblocks > kNoAllocMaxBlocks || gy > 65535 || gz > 65535) {
        char msg[256];
        std::snprintf(msg, sizeof(msg),
                      "homg_residual_norm_noalloc: this grid needs %lld per-block partials, the static scratch holds %d "
                      "(ceil(nx/32) * ceil(ny/8) * nz must not exceed it; e.g. up to 257^3 or 4097^2): use a homg_solver",
                      nblocks, kNoAllocMaxBlocks);
        return fail(HOMG_EINVAL, err, err_cap, msg);
    }
    double* partial = nullptr;
    int dev = 0;
    cudaError_t e = scratch_address(&partial, &dev);
    if (e == cudaSuccess) {
        const dim3 grid((unsigned)gx, (unsigned)gy, (unsigned)gz);
        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        if (dtype == HOMG_F32) e = ndim == 2 ? run<float, 2>(g, h, u_dev, f_dev, partial, int(nblocks), grid, norm_out_dev, st)
                                            : run<float, 3>(g, h, u_dev, f_dev, partial, int(nblocks), grid, norm_out_dev, st);
        else e = ndim == 2 ? run<double, 2>(g, h, u_dev, f_dev, partial, int(nblocks), grid, norm_out_dev, st)
                           : run<double, 3>(g, h, u_dev, f_dev, partial, int(nblocks), grid, norm_out_dev, st);
    }
    if (e != cudaSuccess) {
        char msg[256];
        std::snprintf(msg, sizeof(msg), "homg_residual_norm_noalloc: %s", cudaGetErrorString(e));
        return fail(HOMG_ECUDA, err, err_cap, msg);
    }
    return HOMG_OK;
}
