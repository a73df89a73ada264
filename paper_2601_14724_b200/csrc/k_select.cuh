// a2 + a3 + a4 + a6 fused, one thread block per (stream, layer):
//   a2  A = alpha W (Eq. 2), R = alpha exp(-k (T-1-i)) (Eq. 1), S = (1-w) A + w R (Eq. 3-4)
//   a3  S~^l = (1-lam) S^l + lam S^{l+1} (Eq. 5, raw S^{l+1}; lam of Eq. 7)
//   a4  I_l = TopK(S~^l, |M|) (Eq. 6): radix select of the T-|M| smallest under the total order
//       (score, index) -- ties evict the smaller index -- then a flag scan that emits I_l ascending
//   a6  new positions (Eq. 8: offset + rank; Eq. 11: per-axis rank among DISTINCT retained coordinates)
// Scores live in shared memory for the whole block; W^l and W^{l+1} are re-read from L2.
#pragma once
#include "common.cuh"

namespace hk {

constexpr int kSelThreads = 1024;
constexpr int kBitmapWords = 2048;                   // 65536 coordinate values per axis

__device__ inline uint32_t orderable(float f) {      // monotone float -> uint32 map
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// Exclusive scan of one int per thread over the block (1024 threads); returns the prefix, writes total.
__device__ inline int block_exscan(int v, int* warp_tot /*[33]*/, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int n = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += n;
  }
  __syncthreads();                                   // protect warp_tot from the previous use
  if (lane == 31) warp_tot[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = warp_tot[lane], winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int n = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += n;
    }
    warp_tot[lane] = winc - w;
    if (lane == 31) warp_tot[32] = winc;
  }
  __syncthreads();
  *total = warp_tot[32];
  return warp_tot[warp] + inc - v;
}

__device__ inline float block_reduce_max(float v, float* scratch /*[32]*/) {
  v = warp_max(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  float r = scratch[threadIdx.x & 31];
  return warp_max(r);
}
__device__ inline float block_reduce_sum(float v, float* scratch) {
  v = warp_sum(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  float r = scratch[threadIdx.x & 31];
  return warp_sum(r);
}
__device__ inline int block_reduce_min_i(int v, int* scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, o));
  __syncthreads();
  if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  int r = scratch[threadIdx.x & 31];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) r = min(r, __shfl_xor_sync(0xffffffffu, r, o));
  return r;
}

// W of one layer at token i: per-KV-head column sums added in fixed head order, / (Hq * P).
__device__ inline float mean_w(const Geom& g, int bl, int i, float inv_rows, int n_vh) {
  const float* c = g.colsum + size_t(bl) * g.n_vh_max * g.cap + i;
  float w = 0.f;
  for (int h = 0; h < n_vh; ++h) w += c[size_t(h) * g.cap];
  return w * inv_rows;
}

__global__ void __launch_bounds__(kSelThreads)
k_select(Geom g, int cur, int Tn, int P, float k_forget, int norm_sum, float r_norm_sum, int n_vh) {
  extern __shared__ float s_sc[];                    // [Tn] smoothed scores
  __shared__ int hist[256];
  __shared__ int warp_tot[33];
  __shared__ float red_f[32];
  __shared__ int red_i[32];
  __shared__ uint32_t bitmap[kBitmapWords];
  __shared__ int word_prefix[kBitmapWords];
  __shared__ uint32_t sel_prefix;
  __shared__ int sel_remaining;

  const int bl = blockIdx.x, l = bl % g.L;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool scored0 = l >= g.n_shallow;
  const bool has_next = l + 1 < g.L;
  const bool scored1 = has_next && (l + 1 >= g.n_shallow);
  const float inv_rows = 1.0f / float(g.Hq * P);

  // ---- a2: per-layer normalisation factor alpha (max or sum of W) ------------------------------
  float n0 = 0.f, n1 = 0.f;
  for (int i = tid; i < Tn; i += kSelThreads) {
    if (scored0) { const float w = mean_w(g, bl, i, inv_rows, n_vh); n0 = norm_sum ? n0 + w : fmaxf(n0, w); }
    if (scored1) { const float w = mean_w(g, bl + 1, i, inv_rows, n_vh); n1 = norm_sum ? n1 + w : fmaxf(n1, w); }
  }
  n0 = norm_sum ? block_reduce_sum(n0, red_f) : block_reduce_max(n0, red_f);
  n1 = norm_sum ? block_reduce_sum(n1, red_f) : block_reduce_max(n1, red_f);
  const float a0 = scored0 ? 1.0f / n0 : 0.f, a1 = scored1 ? 1.0f / n1 : 0.f;
  const float om0 = g.omega[l], om1 = has_next ? g.omega[l + 1] : 0.f;
  const float lam = has_next ? g.lambda[l] : 0.f;
  const float r_norm = norm_sum ? r_norm_sum : 1.0f;

  // ---- a2/a3: S^l, S^{l+1}, S~^l ---------------------------------------------------------------
  float* scores_out = g.scores + size_t(bl) * g.cap;
  for (int i = tid; i < Tn; i += kSelThreads) {
    const float R = expf(-k_forget * float(Tn - 1 - i)) * r_norm;           // Eq. 1
    const float A0 = scored0 ? mean_w(g, bl, i, inv_rows, n_vh) * a0 : 0.f;       // Eq. 2
    float s = (1.0f - om0) * A0 + om0 * R;                                   // Eq. 4
    if (has_next) {
      const float A1 = scored1 ? mean_w(g, bl + 1, i, inv_rows, n_vh) * a1 : 0.f;
      const float s1 = (1.0f - om1) * A1 + om1 * R;
      s = (1.0f - lam) * s + lam * s1;                                       // Eq. 5
    }
    s_sc[i] = s;
    scores_out[i] = s;
  }
  __syncthreads();

  // ---- a4: radix select of the E-th smallest key (8 bits per round, MSB first) ------------------
  const int E = Tn - g.budget;
  if (tid == 0) { sel_prefix = 0u; sel_remaining = E; }
  for (int round = 0; round < 4; ++round) {
    const int shift = 24 - 8 * round;
    const uint32_t himask = round == 0 ? 0u : (0xFFFFFFFFu << (shift + 8));
    if (tid < 256) hist[tid] = 0;
    __syncthreads();
    const uint32_t prefix = sel_prefix;
    for (int i0 = 0; i0 < Tn; i0 += kSelThreads) {     // whole warps iterate together
      const int i = i0 + tid;
      uint32_t digit = 0xFFFFFFFFu;
      if (i < Tn) {
        const uint32_t key = orderable(s_sc[i]);
        if ((key & himask) == prefix) digit = (key >> shift) & 255u;
      }
      const uint32_t peers = __match_any_sync(0xffffffffu, digit);            // warp-aggregated histogram
      if (digit != 0xFFFFFFFFu && lane == __ffs(peers) - 1) atomicAdd(&hist[digit], __popc(peers));
    }
    __syncthreads();
    if (warp == 0) {                                    // find the bucket holding the E-th smallest
      int c[8], tot = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) { c[j] = hist[lane * 8 + j]; tot += c[j]; }
      int inc = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
      }
      const int rem = sel_remaining;
      __syncwarp();                                     // every lane has read rem before one lane rewrites it
      int below = inc - tot;                            // candidates in buckets before this lane's 8
      if (below < rem && rem <= inc) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          if (below < rem && rem <= below + c[j]) {
            sel_prefix = prefix | (uint32_t(lane * 8 + j) << shift);
            sel_remaining = rem - below;
          }
          below += c[j];
        }
      }
    }
    __syncthreads();
  }
  const uint32_t vstar = sel_prefix;                    // key of the E-th smallest score
  const int r_eq = sel_remaining;                       // evicted among keys == vstar (smallest indices)

  // ---- flags + scans: thread t owns the contiguous tokens [t*per, (t+1)*per) --------------------
  const int per = (Tn + kSelThreads - 1) / kSelThreads;
  const int i_beg = min(tid * per, Tn), i_end = min(i_beg + per, Tn);
  int n_eq = 0;
  for (int i = i_beg; i < i_end; ++i) n_eq += (orderable(s_sc[i]) == vstar);
  int tot_eq;
  int eq_before = block_exscan(n_eq, warp_tot, &tot_eq);
  int n_keep = 0;
  for (int i = i_beg; i < i_end; ++i) {
    const uint32_t key = orderable(s_sc[i]);
    const bool evict = key < vstar || (key == vstar && eq_before < r_eq);
    eq_before += (key == vstar);
    n_keep += !evict;
  }
  int tot_keep;
  int out = block_exscan(n_keep, warp_tot, &tot_keep);
  int32_t* kept = g.kept + size_t(bl) * g.budget;
  eq_before = block_exscan(n_eq, warp_tot, &tot_eq);    // recompute the prefix consumed above
  for (int i = i_beg; i < i_end; ++i) {
    const uint32_t key = orderable(s_sc[i]);
    const bool evict = key < vstar || (key == vstar && eq_before < r_eq);
    eq_before += (key == vstar);
    if (!evict) kept[out++] = i;
  }
  __syncthreads();                                      // kept[] visible to the whole block

  // ---- a6: new positions into the other buffer ---------------------------------------------------
  const int32_t* pos_old = g.posc + (size_t(bl) * 2 + cur) * g.n_axes * g.cap;
  int32_t* pos_new = g.posc + (size_t(bl) * 2 + (cur ^ 1)) * g.n_axes * g.cap;
  if (g.n_axes == 1) {                                  // Eq. 8: positions increase with the index -> rank = slot
    int32_t* dl = g.delta + size_t(bl) * g.budget;
    for (int s = tid; s < g.budget; s += kSelThreads) {
      pos_new[s] = g.pos_offset + s;
      dl[s] = g.pos_offset + s - pos_old[kept[s]];
    }
    return;
  }
  for (int a = 0; a < 3; ++a) {
    const int32_t* po = pos_old + size_t(a) * g.cap;
    int32_t* pn = pos_new + size_t(a) * g.cap;
    int32_t* dl = g.delta + (size_t(bl) * 3 + a) * g.budget;
    if (!((g.compact_axes >> a) & 1)) {                 // axis kept as is (DESIGN c13)
      for (int s = tid; s < g.budget; s += kSelThreads) { pn[s] = po[kept[s]]; dl[s] = 0; }
      continue;
    }
    int vmin = INT_MAX, vmax_neg = INT_MAX;
    for (int s = tid; s < g.budget; s += kSelThreads) {
      const int v = po[kept[s]];
      vmin = min(vmin, v); vmax_neg = min(vmax_neg, -v);
    }
    vmin = block_reduce_min_i(vmin, red_i);
    const int vmax = -block_reduce_min_i(vmax_neg, red_i);
    if (vmax - vmin >= kBitmapWords * 32) {             // cannot rank: report, leave the axis untouched
      if (tid == 0) atomicOr(g.status, 1);
      for (int s = tid; s < g.budget; s += kSelThreads) { pn[s] = po[kept[s]]; dl[s] = 0; }
      continue;
    }
    for (int w = tid; w < kBitmapWords; w += kSelThreads) bitmap[w] = 0u;
    __syncthreads();
    for (int s = tid; s < g.budget; s += kSelThreads) {
      const int v = po[kept[s]] - vmin;
      atomicOr(&bitmap[v >> 5], 1u << (v & 31));
    }
    __syncthreads();
    const int pc = __popc(bitmap[2 * tid]) + __popc(bitmap[2 * tid + 1]);   // 2 words per thread
    int tot;
    const int pre = block_exscan(pc, warp_tot, &tot);
    word_prefix[2 * tid] = pre;
    word_prefix[2 * tid + 1] = pre + __popc(bitmap[2 * tid]);
    __syncthreads();
    for (int s = tid; s < g.budget; s += kSelThreads) {  // Eq. 11: offset + rank among distinct coordinates
      const int v = po[kept[s]] - vmin;
      const int p_new = g.pos_offset + word_prefix[v >> 5] + __popc(bitmap[v >> 5] & ((1u << (v & 31)) - 1u));
      pn[s] = p_new;
      dl[s] = p_new - (v + vmin);
    }
    __syncthreads();
  }
}

}  // namespace hk
