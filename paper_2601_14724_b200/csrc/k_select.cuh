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

// a2 (first half), fully parallel: W_i = per-(KV head, super-chunk) column sums added in fixed order /
// (Hq * P), and the per-layer max of W (order-independent, so an atomic max keeps it deterministic).
__global__ void __launch_bounds__(256)
k_wsum(Geom g, int Tn, int P, int n_vh) {
  __shared__ float red[8];
  pdl_wait();
  pdl_launch_dependents();
  const int Ls = g.L - g.n_shallow;
  const int bl = (blockIdx.y / Ls) * g.L + g.n_shallow + blockIdx.y % Ls;
  const int i = blockIdx.x * 256 + threadIdx.x;
  Tn = layer_T(g, bl % g.L, Tn);
  float w = 0.f;
  if (i < Tn) {
    const float* c = g.colsum + size_t(bl) * g.n_vh_max * g.cap + i;
    for (int h = 0; h < n_vh; ++h) w += __ldcg(c + size_t(h) * g.cap);
    const int l = bl % g.L;
    const int p_eff = l >= g.L - g.n_deep ? P - g.probe_deep_begin : P;    // deep layers: global-prompt rows only
    w *= 1.0f / float(g.Hq * p_eff);
    g.wsum[size_t(bl) * g.cap + i] = w;
  }
  const float m = warp_max(w);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x < 32) {
    float r = threadIdx.x < 8 ? red[threadIdx.x] : 0.f;
    r = warp_max(r);
    if (threadIdx.x == 0) atomicMax(&g.wmax[bl], __float_as_uint(r));
  }
}

__global__ void __launch_bounds__(kSelThreads)
k_select(Geom g, int cur, int Tn, float k_forget, int norm_sum, float r_norm_sum, int reindex, int summary_pos) {
  extern __shared__ float s_sc[];                    // [Tn] smoothed scores
  // per-warp digit histograms (radix phase); the M-RoPE rank bitmap + word prefixes reuse the space later
  __shared__ __align__(16) int whist[32 * 256];
  __shared__ int part[4][256];
  __shared__ int warp_tot[33];
  __shared__ float red_f[32];
  __shared__ int red_i[32];
  __shared__ uint32_t sel_prefix;
  __shared__ int sel_remaining;
  uint32_t* bitmap = reinterpret_cast<uint32_t*>(whist);              // [kBitmapWords]
  int* word_prefix = whist + kBitmapWords;                            // [kBitmapWords]

  pdl_wait();
  pdl_launch_dependents();
  const int bl = blockIdx.x, l = bl % g.L;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // layer-dependent budgets (DESIGN f4): this layer's own candidates and budget; Eq. 5 pairs candidate i with candidate
  // i + shift1 of layer l + 1 (equal distance from the newest token), candidates without a counterpart keep S^l
  const int T1 = l + 1 < g.L ? layer_T(g, l + 1, Tn) : Tn;
  Tn = layer_T(g, l, Tn);
  const int shift1 = T1 - Tn;
  const int budget_l = layer_keep(g, l);
  const bool scored0 = l >= g.n_shallow;
  const bool has_next = l + 1 < g.L;
  const bool scored1 = has_next && (l + 1 >= g.n_shallow);

  // ---- a2: per-layer normalisation factor alpha (max or sum of W) ------------------------------
  const float* w0 = g.wsum + size_t(bl) * g.cap;
  const float* w1 = w0 + g.cap;
  float n0, n1;
  if (norm_sum) {
    float t0 = 0.f, t1 = 0.f;
    for (int i = tid; i < max(Tn, T1); i += kSelThreads) { if (scored0 && i < Tn) t0 += __ldcg(w0 + i); if (scored1 && i < T1) t1 += __ldcg(w1 + i); }
    n0 = block_reduce_sum(t0, red_f);
    n1 = block_reduce_sum(t1, red_f);
  } else {
    n0 = scored0 ? __uint_as_float(__ldcg(g.wmax + bl)) : 1.f;
    n1 = scored1 ? __uint_as_float(__ldcg(g.wmax + bl + 1)) : 1.f;
  }
  const float a0 = scored0 ? 1.0f / n0 : 0.f, a1 = scored1 ? 1.0f / n1 : 0.f;
  const float om0 = g.omega[l], om1 = has_next ? g.omega[l + 1] : 0.f;
  const float lam = has_next ? g.lambda[l] : 0.f;
  float r_norm = norm_sum ? r_norm_sum : 1.0f, r_norm1 = r_norm;
  if (norm_sum && g.lay_T) {                         // layer-dependent budgets: each layer's recency sums over its own T
    r_norm = float((1.0 - exp(-double(k_forget))) / (1.0 - exp(-double(k_forget) * Tn)));
    r_norm1 = float((1.0 - exp(-double(k_forget))) / (1.0 - exp(-double(k_forget) * T1)));
  }
  // ---- a2/a3: S^l, S^{l+1}, S~^l (4 tokens per thread per trip: all loads issued before use) ----
  float* scores_out = g.scores + size_t(bl) * g.cap;
  for (int i0 = tid; i0 < Tn; i0 += 4 * kSelThreads) {
    float x0[4], x1[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int i = i0 + j * kSelThreads;
      x0[j] = (scored0 && i < Tn) ? __ldcg(w0 + i) : 0.f;
      x1[j] = (scored1 && i < Tn && i + shift1 >= 0) ? __ldcg(w1 + i + shift1) : 0.f;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int i = i0 + j * kSelThreads;
      if (i < Tn) {
        const float e = expf(-k_forget * float(Tn - 1 - i));                 // Eq. 1
        const float R = e * r_norm;
        float sc = (1.0f - om0) * (x0[j] * a0) + om0 * R;                    // Eq. 2, Eq. 4
        if (has_next && i + shift1 >= 0) {
          const float s1 = (1.0f - om1) * (x1[j] * a1) + om1 * (e * r_norm1);
          sc = (1.0f - lam) * sc + lam * s1;                                 // Eq. 5
        }
        s_sc[i] = sc;
        scores_out[i] = sc;
      }
    }
  }
  // deep layers of a summary-token cache keep one token fewer: slot budget-1 is the summary token (DESIGN f1)
  const bool summ = g.summary && l >= g.L - g.n_deep;
  const int n_keep = budget_l - (summ ? 1 : 0);
  if (budget_l >= Tn) {
    // layer-dependent budgets: this layer is under its budget at this arrival -- nothing is evicted, nothing re-indexed
    // (1D RoPE only, validated at create); the gather then copies every row as it is
    const int32_t* po = g.posc + (size_t(bl) * 2 + cur) * g.n_axes * g.cap;
    int32_t* pn = g.posc + (size_t(bl) * 2 + (cur ^ 1)) * g.n_axes * g.cap;
    for (int i = tid; i < Tn; i += kSelThreads) {
      g.kept[size_t(bl) * g.budget + i] = i;
      g.delta[size_t(bl) * g.n_axes * g.budget + i] = 0;
      pn[i] = __ldcg(po + i);
    }
    return;
  }
  if (tid == 0) { sel_prefix = 0u; sel_remaining = Tn - n_keep; }
  for (int i = tid; i < 32 * 256; i += kSelThreads) whist[i] = 0;
  __syncthreads();
  // ---- a4: radix select of the E-th smallest key (8 bits per round, MSB first) ------------------
  for (int round = 0; round < 4; ++round) {
    const int shift = 24 - 8 * round;
    const uint32_t himask = round == 0 ? 0u : (0xFFFFFFFFu << (shift + 8));
    const uint32_t prefix = sel_prefix;
    int* my_hist = whist + warp * 256;
    for (int i0 = 0; i0 < Tn; i0 += kSelThreads) {     // whole warps iterate together
      const int i = i0 + tid;
      uint32_t digit = 0xFFFFFFFFu;
      if (i < Tn) {
        const uint32_t key = orderable(s_sc[i]);
        if ((key & himask) == prefix) digit = (key >> shift) & 255u;
      }
      // warp-private histogram: the shared-memory atomics only ever collide inside one warp (aggregating equal digits with
      // __match_any_sync first, one add per group, measured slower: wsum + select 24 -> 30 us, 59 -> 91 us at T = 32 964)
      if (digit != 0xFFFFFFFFu) atomicAdd(&my_hist[digit], 1);
    }
    __syncthreads();
    {                                                   // fold 8 warp histograms per thread (4 partial sums per digit),
      const int q = tid >> 8, d = tid & 255;            // clearing them for the next round
      int c = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) { c += whist[(q * 8 + w) * 256 + d]; whist[(q * 8 + w) * 256 + d] = 0; }
      part[q][d] = c;
    }
    __syncthreads();
    if (warp == 0) {                                    // find the bucket holding the E-th smallest
      int c[8], tot = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int d = lane * 8 + j;
        c[j] = (part[0][d] + part[1][d]) + (part[2][d] + part[3][d]);
        tot += c[j];
      }
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

  // ---- flags + one packed scan over 32-token chunks; outputs are written coalesced -------------
  // evicted(i) = key < v*  or  (key == v* and fewer than r_eq equal keys precede i)
  // chunk c = tokens [32c, 32c+32): cnt_c = #(key < v*) | #(key == v*) << 16, exclusive-scanned over c.
  const int n_chunks = (Tn + 31) >> 5;                                   // <= 1024 * kChunkPerThread
  int* chunk_pre = whist;                                                // reuse: [n_chunks] packed prefixes
  for (int c = warp; c < n_chunks; c += 32) {
    const int i = c * 32 + lane;
    const uint32_t key = i < Tn ? orderable(s_sc[i]) : 0xFFFFFFFFu;
    const uint32_t lt = __ballot_sync(0xffffffffu, i < Tn && key < vstar);
    const uint32_t eq = __ballot_sync(0xffffffffu, i < Tn && key == vstar);
    if (lane == 0) chunk_pre[c] = __popc(lt) | (__popc(eq) << 16);
  }
  __syncthreads();
  {
    const int cpt = (n_chunks + kSelThreads - 1) / kSelThreads;          // chunks per thread (1 up to 32K tokens)
    const int c_beg = min(tid * cpt, n_chunks), c_end = min(c_beg + cpt, n_chunks);
    int mine = 0;
    for (int c = c_beg; c < c_end; ++c) mine += chunk_pre[c];
    int tot;
    int run = block_exscan(mine, warp_tot, &tot);                        // both halves stay < 65536
    for (int c = c_beg; c < c_end; ++c) { const int v = chunk_pre[c]; chunk_pre[c] = run; run += v; }
  }
  __syncthreads();
  int32_t* kept = g.kept + size_t(bl) * g.budget;
  const int32_t* pos_old = g.posc + (size_t(bl) * 2 + cur) * g.n_axes * g.cap;
  int32_t* pos_new = g.posc + (size_t(bl) * 2 + (cur ^ 1)) * g.n_axes * g.cap;
  int32_t* dl1 = g.delta + size_t(bl) * g.n_axes * g.budget;
  const uint32_t lane_lt = (1u << lane) - 1u;
  for (int cb = warp; cb < n_chunks; cb += 32 * 8) {                     // 8 chunks per trip: old positions first
    int p_old[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int i = (cb + 32 * j) * 32 + lane;
      p_old[j] = (g.n_axes == 1 && i < Tn) ? __ldcg(pos_old + i) : 0;
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int c = cb + 32 * j;                                         // warp-uniform
      if (c >= n_chunks) break;
      const int i = c * 32 + lane;
      const uint32_t key = i < Tn ? orderable(s_sc[i]) : 0xFFFFFFFFu;
      const uint32_t lt = __ballot_sync(0xffffffffu, i < Tn && key < vstar);
      const uint32_t eq = __ballot_sync(0xffffffffu, i < Tn && key == vstar);
      const int pre = chunk_pre[c];
      const int lt_before = (pre & 0xFFFF) + __popc(lt & lane_lt);
      const int eq_before = (pre >> 16) + __popc(eq & lane_lt);
      const bool evict = key < vstar || (key == vstar && eq_before < r_eq);
      if (summ && i < Tn && evict) g.evicted[size_t(bl) * g.n_evict_max + lt_before + min(eq_before, r_eq)] = i;
      if (i < Tn && !evict) {
        const int out = i - lt_before - min(eq_before, r_eq);            // slot of token i among the kept
        kept[out] = i;
        if (g.n_axes == 1) {                                             // Eq. 8: positions rise with the index -> rank = slot
          // lazy mode between re-index steps keeps the original index: delta 0 = bit-exact key copy
          pos_new[out] = reindex ? g.pos_offset + out : p_old[j];
          dl1[out] = reindex ? g.pos_offset + out - p_old[j] : 0;
        }
      }
    }
  }
  if (summ && tid == 0) {                               // the summary token's slot (filled by k_summary)
    kept[n_keep] = -1; pos_new[n_keep] = reindex ? g.pos_offset + n_keep : summary_pos; dl1[n_keep] = 0;
  }
  if (g.n_axes == 1) return;
  __syncthreads();                                      // kept[] visible to the whole block

  // ---- a6 (M-RoPE): per-axis rank among the distinct retained coordinates (Eq. 11) ----------------
  for (int a = 0; a < 3; ++a) {
    const int32_t* po = pos_old + size_t(a) * g.cap;
    int32_t* pn = pos_new + size_t(a) * g.cap;
    int32_t* dl = g.delta + (size_t(bl) * 3 + a) * g.budget;
    if (!reindex || !((g.compact_axes >> a) & 1)) {     // axis kept as is (DESIGN c13; lazy mode between re-index steps)
      for (int s = tid; s < g.budget; s += kSelThreads) { pn[s] = __ldcg(po + kept[s]); dl[s] = 0; }
      continue;
    }
    int vmin = INT_MAX, vmax_neg = INT_MAX;
    for (int s = tid; s < g.budget; s += kSelThreads) {
      const int v = __ldcg(po + kept[s]);
      vmin = min(vmin, v); vmax_neg = min(vmax_neg, -v);
    }
    vmin = block_reduce_min_i(vmin, red_i);
    const int vmax = -block_reduce_min_i(vmax_neg, red_i);
    if (vmax - vmin >= kBitmapWords * 32) {             // cannot rank: report, leave the axis untouched
      if (tid == 0) atomicOr(g.status, 1);
      for (int s = tid; s < g.budget; s += kSelThreads) { pn[s] = __ldcg(po + kept[s]); dl[s] = 0; }
      continue;
    }
    __syncthreads();
    for (int w = tid; w < kBitmapWords; w += kSelThreads) bitmap[w] = 0u;
    __syncthreads();
    for (int s = tid; s < g.budget; s += kSelThreads) {
      const int v = __ldcg(po + kept[s]) - vmin;
      atomicOr(&bitmap[v >> 5], 1u << (v & 31));
    }
    __syncthreads();
    const int pc = __popc(bitmap[2 * tid]) + __popc(bitmap[2 * tid + 1]);   // 2 words per thread
    int tot;
    const int wpre = block_exscan(pc, warp_tot, &tot);
    word_prefix[2 * tid] = wpre;
    word_prefix[2 * tid + 1] = wpre + __popc(bitmap[2 * tid]);
    __syncthreads();
    for (int s = tid; s < g.budget; s += kSelThreads) {
      const int v = __ldcg(po + kept[s]) - vmin;
      const int p_new = g.pos_offset + word_prefix[v >> 5] + __popc(bitmap[v >> 5] & ((1u << (v & 31)) - 1u));
      pn[s] = p_new;
      dl[s] = p_new - (v + vmin);
    }
    __syncthreads();
  }
}

}  // namespace hk
