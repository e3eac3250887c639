// homg_exec.h — entry points of the cycle executor (internal).
#pragma once
#include "homg_internal.h"

namespace homg {

// kernel classes reported by homg_profile_cycles (order = include/homg.h HOMG_TAG_*)
enum {
    TAG_RESIDUAL0 = 0, TAG_NORM_FINISH, TAG_RESTRICT, TAG_RELAX0, TAG_RELAX, TAG_DELIVER0, TAG_DELIVER,
    TAG_INJECT, TAG_D0, TAG_COARSE, TAG_OTHER, TAG_RELAX0_FIRST, TAG_RELAX0_LAST, TAG_VISIT0, TAG_VISIT, TAG_COUNT
};

constexpr long long kTiledMinNodesDefault = 300000;   // 129^3 and up, 1025^2 and up (65^3 and 513^2 measured faster on the generic kernels)

// Device queries, the driver's tensor-map encoder, kernel attributes.  Called once by homg_create.
cudaError_t exec_init(homg_solver* s);

// measured on cfg2 (profiles/): one-CTA runs pay off up to 9^3; a 17^3 / 33^3 operation needs more load
// bandwidth than a few SMs have, so those levels keep one launch per operation
constexpr long long kCoarseNodesDefault = 800;

// Builds the coarse-level program of one cycle (planning pass, no launches) and uploads it to a
// small library-owned device buffer.  Must run before exec_cycle and outside stream capture.
cudaError_t exec_prepare(homg_solver* s);

// Issues the launches of ONE outer cycle on `st` (which may be a capturing stream) and fills
// s->launches_per_cycle / s->bytes_cycle_*.
cudaError_t exec_cycle(homg_solver* s, cudaStream_t st);
// homg_solve: the launches of the prologue (S1 of the initial guess) and of the loop body (S2..S4, then S1 of the
// new u) of the device-side WHILE loop; `cond` is the cudaGraphConditionalHandle the norm kernel sets.
cudaError_t exec_solve_prologue(homg_solver* s, cudaStream_t st, unsigned long long cond);
cudaError_t exec_solve_body(homg_solver* s, cudaStream_t st, unsigned long long cond);
// One cycle with plain stream launches, an event after every launch; accumulates the elapsed ms and
// launch counts per TAG_* (arrays of TAG_COUNT).  Synchronises the stream.
cudaError_t exec_cycle_profiled(homg_solver* s, cudaStream_t st, double* ms_by_tag, int* launches_by_tag,
                                double* bytes_by_tag);
// ||f - A u||^2 of the current u -> *s->scalar (no history entry).
cudaError_t exec_norm_only(homg_solver* s, cudaStream_t st);
// mixed precision: nodal k of the fp64 outer problem -> fp32 k of the inner hierarchy (level 0)
cudaError_t exec_cvt_coef_to_inner(homg_solver* s, cudaStream_t st);
// k_m = k_{m-1} sampled at even nodes, m = 1..M.
cudaError_t exec_sample_coef(homg_solver* s, cudaStream_t st);
// dense C-order device array <-> padded level-0 array.
cudaError_t exec_pack(homg_solver* s, cudaStream_t st, const void* dense_dev, void* padded, int zero_boundary);
cudaError_t exec_unpack(homg_solver* s, cudaStream_t st, const void* padded, void* dense_dev);

}  // namespace homg
