// a1 -- attention importance W (Eq. 2), CUDA-core path.
//
// W_i = mean over query heads h and probe rows r of softmax_i(scale * q_{h,r} . k_{i,h/G}).
// The softmax normaliser of a probe row needs every token, the column sum of a token needs every
// row, so the contraction runs twice (flash-style recompute, nothing T x R is ever stored):
//   pass 1 (kStats)  : per probe row, partial (max, sum exp) over each 128-token tile -> `partial`
//   combine          : per probe row, (m, 1/Z) over all tiles                         -> `rowstat`
//   pass 2 (kColsum) : per token, sum_r exp(s - m_r) / Z_r over the rows of one KV head -> `colsum`
// All in fp32, log2 domain (t = s * scale * log2 e, exp2f).  This path serves fp32 caches, small
// head_dim and shapes too small to fill tcgen05 tiles; the dense bf16 case goes to k_score_tc.cuh.
#pragma once
#include "common.cuh"

namespace hk {

constexpr int kSimtTokens = 128;   // tokens per block = threads per block (one token per thread)
constexpr int kSimtRowChunk = 32;  // probe rows staged in shared memory at a time
constexpr int kSimtRowGroup = 8;   // rows accumulated per thread at a time

template <typename T, int D, bool kColsum>
__global__ void __launch_bounds__(kSimtTokens)
k_score_simt(Geom g, const T* __restrict__ q_probe, int cur, int Tn, int P, float scale_log2, int n_part) {
  __shared__ __align__(16) float q_s[kSimtRowChunk][D];
  __shared__ float stat_s[kSimtRowChunk][2];        // pass 2: (m2, 1/Z) of the staged rows
  __shared__ float part_s[4][kSimtRowChunk][2];     // pass 1: per-warp (m2, z)

  const int Ls = g.L - g.n_shallow;
  const int b = blockIdx.z / Ls, l = g.n_shallow + blockIdx.z % Ls;
  const int bl = b * g.L + l;
  const int kvh = blockIdx.y;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tok = blockIdx.x * kSimtTokens + tid;
  const bool valid = tok < layer_T(g, l, Tn);      // layer-dependent budgets: blocks past T_l contribute (-inf, 0) / nothing
  const int R = g.G * P;                             // probe rows sharing this KV head (contiguous in Q)
  const int row0 = kvh * R;                          // first of them within the layer's Hq*P rows

  // this thread's key, widened to fp32 registers
  float kreg[D];
  {
    const T* krow = reinterpret_cast<const T*>(g.kc) +
                    ((size_t(bl) * 2 + cur) * g.cap + (valid ? tok : 0)) * g.row_elems + kvh * D;
    constexpr int V = Elem<T>::kPerVec;
#pragma unroll
    for (int c = 0; c < D; c += V) {
      uint4 v = *reinterpret_cast<const uint4*>(krow + c);
      Elem<T>::unpack(v, &kreg[c]);
    }
  }
  const T* qg = q_probe + (size_t(bl) * g.Hq * P + row0) * D;
  const float* rowstat = g.rowstat + (size_t(bl) * g.Hq * g.p_max + row0) * 2;
  float acc_w = 0.f;

  for (int r0 = 0; r0 < R; r0 += kSimtRowChunk) {
    __syncthreads();
    for (int i = tid; i < kSimtRowChunk * D; i += kSimtTokens) {
      const int rr = i / D, c = i % D;
      q_s[rr][c] = (r0 + rr < R) ? Elem<T>::to_float(qg[size_t(r0 + rr) * D + c]) : 0.f;
    }
    if (kColsum && tid < kSimtRowChunk) {
      // deep layers ignore the local-prompt rows (probe index < probe_deep_begin) of every query head
      const bool ok = r0 + tid < R && !(l >= g.L - g.n_deep && (r0 + tid) % P < g.probe_deep_begin);
      stat_s[tid][0] = ok ? rowstat[(r0 + tid) * 2] : 0.f;
      stat_s[tid][1] = ok ? rowstat[(r0 + tid) * 2 + 1] : 0.f;   // 1/Z = 0 masks rows past R
    }
    __syncthreads();
#pragma unroll 1
    for (int rr = 0; rr < kSimtRowChunk; rr += kSimtRowGroup) {
      float acc[kSimtRowGroup];
#pragma unroll
      for (int i = 0; i < kSimtRowGroup; ++i) acc[i] = 0.f;
#pragma unroll
      for (int c = 0; c < D; c += 4) {
#pragma unroll
        for (int i = 0; i < kSimtRowGroup; ++i) {
          const float4 q4 = *reinterpret_cast<const float4*>(&q_s[rr + i][c]);   // warp-broadcast
          acc[i] = fmaf(kreg[c], q4.x, acc[i]);
          acc[i] = fmaf(kreg[c + 1], q4.y, acc[i]);
          acc[i] = fmaf(kreg[c + 2], q4.z, acc[i]);
          acc[i] = fmaf(kreg[c + 3], q4.w, acc[i]);
        }
      }
#pragma unroll
      for (int i = 0; i < kSimtRowGroup; ++i) {
        const float t = valid ? acc[i] * scale_log2 : -INFINITY;
        if (kColsum) {
          acc_w = fmaf(exp2f(t - stat_s[rr + i][0]), stat_s[rr + i][1], acc_w);
        } else {
          const float m = warp_max(t);
          const float e = (m == -INFINITY) ? 0.f : exp2f(t - m);
          const float z = warp_sum(e);
          if (lane == 0) { part_s[warp][rr + i][0] = m; part_s[warp][rr + i][1] = z; }
        }
      }
    }
    if (!kColsum) {
      __syncthreads();
      if (tid < kSimtRowChunk && r0 + tid < R) {      // merge the 4 warps' (m, z) of row r0 + tid
        float m = -INFINITY;
#pragma unroll
        for (int w = 0; w < 4; ++w) m = fmaxf(m, part_s[w][tid][0]);
        float z = 0.f;
#pragma unroll
        for (int w = 0; w < 4; ++w)
          z += (part_s[w][tid][0] == -INFINITY) ? 0.f : part_s[w][tid][1] * exp2f(part_s[w][tid][0] - m);
        float* out = g.partial + ((size_t(bl) * g.Hq * g.p_max + row0 + r0 + tid) * n_part + blockIdx.x) * 2;
        out[0] = m; out[1] = z;
      }
    }
  }
  if (kColsum && valid) g.colsum[(size_t(bl) * g.n_vh_max + kvh) * g.cap + tok] = acc_w;
}

// Per probe row: merge n_part partial (m2, z) into (m2, 1/Z).  One warp per row.
__global__ void __launch_bounds__(256)
k_score_combine(Geom g, int P, int n_part) {
  const int Ls = g.L - g.n_shallow;
  const int rows = g.Hq * P;
  const int warp_global = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp_global >= g.B * Ls * rows) return;
  const int row = warp_global % rows, bls = warp_global / rows;
  const int bl = (bls / Ls) * g.L + g.n_shallow + bls % Ls;
  const float* p = g.partial + (size_t(bl) * g.Hq * g.p_max + row) * n_part * 2;
  float m = -INFINITY;
  for (int i = lane; i < n_part; i += 32) m = fmaxf(m, p[2 * i]);
  m = warp_max(m);
  float z = 0.f;
  for (int i = lane; i < n_part; i += 32) {
    const float mi = p[2 * i];
    z += (mi == -INFINITY) ? 0.f : p[2 * i + 1] * exp2f(mi - m);
  }
  z = warp_sum(z);
  if (lane == 0) {
    float* out = g.rowstat + (size_t(bl) * g.Hq * g.p_max + row) * 2;
    out[0] = m; out[1] = 1.0f / z;
  }
}

}  // namespace hk
