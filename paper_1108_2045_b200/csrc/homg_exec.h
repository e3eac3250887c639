// homg_exec.h — entry points of the cycle executor (internal).
#pragma once
#include "homg_internal.h"

namespace homg {

// Issues the launches of ONE outer cycle on `st` (which may be a capturing stream) and fills
// s->launches_per_cycle / s->bytes_cycle_*.
cudaError_t exec_cycle(homg_solver* s, cudaStream_t st);
// ||f - A u||^2 of the current u -> *s->scalar (no history entry).
cudaError_t exec_norm_only(homg_solver* s, cudaStream_t st);
// k_m = k_{m-1} sampled at even nodes, m = 1..M.
cudaError_t exec_sample_coef(homg_solver* s, cudaStream_t st);
// dense C-order device array <-> padded level-0 array.
cudaError_t exec_pack(homg_solver* s, cudaStream_t st, const void* dense_dev, void* padded, int zero_boundary);
cudaError_t exec_unpack(homg_solver* s, cudaStream_t st, const void* padded, void* dense_dev);

}  // namespace homg
