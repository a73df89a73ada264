// a1 -- attention importance W, tcgen05 / TMEM / TMA path (bf16, head_dim 128).  Placeholder until the
// tensor-core kernels land: reports "unavailable" so AUTO falls back to the CUDA-core path.
#pragma once
#include "host_state.cuh"

namespace hk {
inline bool tc_init(hermes_t* h) { h->err = "tcgen05 path not built"; return false; }
inline void tc_destroy(hermes_t*) {}
inline bool tc_profitable(const hermes_t*, int, int) { return false; }
inline int tc_score(hermes_t*, const void*, int, int, float, cudaStream_t) { return HERMES_ESTATE; }
}  // namespace hk
