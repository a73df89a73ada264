// a0 -- append the arriving chunk to every (stream, layer) slab and assign arrival positions
// (PAPER.md:49, :142).  Pure copy: 128-bit coalesced loads/stores, grid-stride.
#pragma once
#include "common.cuh"

namespace hk {

// K_new/V_new: [B*L][n_new][row_elems]; destination rows [len, len+n_new) of the current buffer.
// row_vecs = 16-byte vectors per token row.  what: bit 0 = K rows + positions + wmax reset, bit 1 = V rows (the host
// entry point appends V in a second launch, after scoring, so that V's host-to-device copy overlaps the scoring).
constexpr int kAppendK = 1, kAppendV = 2;
__global__ void __launch_bounds__(256)
k_append(Geom g, const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
         int cur, int len, int n_new, int row_vecs, int pos_start, int what) {
  pdl_wait();
  pdl_launch_dependents();
  const int bl = blockIdx.y;                        // b * L + l
  if (g.lay_T) len = __ldg(g.lay_T + bl % g.L) - n_new;   // layer-dependent budgets: this layer's own length
  const bool do_k = what & kAppendK, do_v = what & kAppendV;
  if (do_k && blockIdx.x == 0) {                     // per-update counters of this slab: max of W, pass-1 progress of the tcgen05 scoring
    if (threadIdx.x == 0) g.wmax[bl] = 0u;
    for (int i = threadIdx.x; i < g.n_vh_max; i += blockDim.x) g.seg_cnt[size_t(bl) * g.n_vh_max + i] = 0u;
  }
  const size_t slab = size_t(bl) * 2 + cur;
  const size_t n_vec = size_t(n_new) * row_vecs;
  const uint4* ks = k_new + size_t(bl) * n_vec;
  const uint4* vs = v_new + size_t(bl) * n_vec;
  uint4* kd = reinterpret_cast<uint4*>(g.kc) + (slab * g.cap + len) * row_vecs;
  uint4* vd = reinterpret_cast<uint4*>(g.vc) + (slab * g.cap + len) * row_vecs;
  const size_t stride = size_t(gridDim.x) * blockDim.x;
  size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
  // 2 independent (K,V) pairs in flight per thread
  if (do_k && do_v) {
    for (; i + stride < n_vec; i += 2 * stride) {
      uint4 a = ldg_stream(ks + i), b = ldg_stream(vs + i);
      uint4 c = ldg_stream(ks + i + stride), d = ldg_stream(vs + i + stride);
      kd[i] = a; vd[i] = b; kd[i + stride] = c; vd[i + stride] = d;
    }
    if (i < n_vec) { kd[i] = ldg_stream(ks + i); vd[i] = ldg_stream(vs + i); }
  } else {
    const uint4* src = do_k ? ks : vs;
    uint4* dst = do_k ? kd : vd;
    for (; i + stride < n_vec; i += 2 * stride) {
      uint4 a = ldg_stream(src + i), c = ldg_stream(src + i + stride);
      dst[i] = a; dst[i + stride] = c;
    }
    if (i < n_vec) dst[i] = ldg_stream(src + i);
  }
  if (!do_k) return;

  // arrival positions, identical across layers (1D: pos_start + j; M-RoPE: (t0 + j/tpt, grid row, grid col))
  int32_t* pos = g.posc + slab * g.n_axes * g.cap;
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_new; j += gridDim.x * blockDim.x) {
    if (g.n_axes == 1) {
      pos[len + j] = pos_start + j;
    } else {
      const int tpt = g.grid_h * g.grid_w;
      const int r = j % tpt;
      pos[len + j] = pos_start + j / tpt;
      pos[g.cap + len + j] = g.pos_offset + r / g.grid_w;
      pos[2 * g.cap + len + j] = g.pos_offset + r % g.grid_w;
    }
  }
}

}  // namespace hk
