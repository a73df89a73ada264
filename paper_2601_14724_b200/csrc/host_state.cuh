// Host-side state of a handle: validated config, workspace carve-up, host-tracked stream state.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/hermes.h"
#include "common.cuh"

namespace hk {

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct Layout {           // byte offsets into the workspace
  size_t kc, vc, posc, colsum, wsum, wmax, rowstat, partial, scores, kept, delta, evicted, rope_tab, rope_freq, sum_tab, omega, lambda,
      status, seg_cnt, lay_dyn, tc_pre, stage_k, stage_v, stage_q, tmaps, total;
  int cap, n_axes, n_part_max, table_rows, n_shallow, n_middle, n_deep, n_vh_max, sum_tab_neg, sum_tab_rows;
  int budget_max, budget_min;   // largest / smallest layer budget (= budget unless budget_weight is unequal)
  size_t esize, row_bytes, stage_kv_bytes, stage_q_bytes;
};

// Layer-dependent budgets: m_i = floor(w_i / sum_j w_j * budget * L), residue to the last layer; w_i is
// the weight of layer i's stage.  Same arithmetic as the oracle: fp32 weights, left-to-right fp64 sum, fp64 quotient.
inline bool uniform_budgets(const hermes_config& c) {
  return c.budget_weight[0] == c.budget_weight[1] && c.budget_weight[1] == c.budget_weight[2];
}
inline std::vector<int> layer_budgets(const hermes_config& c, int n_shallow, int n_deep) {
  const int L = c.n_layers;
  std::vector<int> m(L, c.budget);
  if (uniform_budgets(c)) return m;
  std::vector<double> w(L);
  double wsum = 0.0;
  for (int l = 0; l < L; ++l) {
    w[l] = double(l < n_shallow ? c.budget_weight[0] : l < L - n_deep ? c.budget_weight[1] : c.budget_weight[2]);
    wsum += w[l];
  }
  const long long total = (long long)c.budget * L;
  long long acc = 0;
  for (int l = 0; l < L; ++l) { m[l] = int(std::floor(w[l] / wsum * double(total))); acc += m[l]; }
  m[L - 1] += int(total - acc);
  return m;
}

inline void stage_split(int L, int& n_shallow, int& n_deep) {   // PAPER.md:144; rounding DESIGN c7
  if (n_shallow < 0) n_shallow = std::max(1, (L + 5) / 10);
  if (n_deep < 0) n_deep = std::max(1, (3 * L + 5) / 10);
}

// Returns nullptr if valid, else a static message.
inline const char* validate(const hermes_config& c) {
  if (c.n_layers <= 0 || c.n_layers > kMaxLayers) return "n_layers out of range [1, 256]";
  if (c.n_q_heads <= 0 || c.n_kv_heads <= 0 || c.n_q_heads % c.n_kv_heads) return "n_q_heads must be a positive multiple of n_kv_heads";
  if (c.head_dim != 32 && c.head_dim != 64 && c.head_dim != 128) return "head_dim must be 32, 64 or 128";
  if (c.dtype != HERMES_F32 && c.dtype != HERMES_BF16) return "dtype must be HERMES_F32 or HERMES_BF16";
  if (c.n_streams <= 0) return "n_streams must be positive";
  if (c.budget <= 0) return "budget must be positive";
  if (c.max_chunk_tokens <= 0) return "max_chunk_tokens must be positive";
  if (c.max_probe_tokens <= 0) return "max_probe_tokens must be positive";
  if (c.max_tokens != 0 && c.max_tokens <= c.budget) return "max_tokens must exceed budget (or be 0)";
  if (!(c.forget_rate > 0.f) || !std::isfinite(c.forget_rate)) return "forget_rate (k of Eq. 1) must be > 0";
  if (c.norm_mode != HERMES_NORM_MAX && c.norm_mode != HERMES_NORM_SUM) return "bad norm_mode";
  int ns = c.n_shallow, nd = c.n_deep;
  stage_split(c.n_layers, ns, nd);
  if (ns < 0 || nd < 0 || ns + nd > c.n_layers) return "n_shallow + n_deep exceeds n_layers";
  if (c.l_short >= 0 && c.l_long >= 0 && c.l_long < c.l_short) return "l_long < l_short";
  const float lam[3] = {c.lambda_shallow, c.lambda_middle, c.lambda_deep};
  for (float v : lam) if (!(v >= 0.f && v <= 1.f)) return "lambda must lie in [0, 1]";
  if (c.softmax_scale < 0.f || !std::isfinite(c.softmax_scale)) return "softmax_scale must be >= 0";
  if (c.rope_mode != HERMES_ROPE_1D && c.rope_mode != HERMES_ROPE_M3D) return "bad rope_mode";
  if (!(c.rope_theta > 0.f)) return "rope_theta must be > 0";
  if (c.rope_mode == HERMES_ROPE_M3D) {
    if (c.mrope_section[0] < 0 || c.mrope_section[1] < 0 || c.mrope_section[2] < 0 ||
        c.mrope_section[0] + c.mrope_section[1] + c.mrope_section[2] != c.head_dim / 2)
      return "mrope_section must sum to head_dim/2";
    if (c.mrope_grid_h <= 0 || c.mrope_grid_w <= 0) return "mrope grid must be positive";
    if (c.mrope_compact_axes < 0 || c.mrope_compact_axes > 7) return "bad mrope_compact_axes";
  }
  if (c.pos_offset < 0) return "pos_offset must be >= 0";
  if (c.reindex_mode != HERMES_REINDEX_EAGER && c.reindex_mode != HERMES_REINDEX_LAZY) return "bad reindex_mode";
  if (c.probe_deep_begin < 0 || c.probe_deep_begin >= c.max_probe_tokens) return "probe_deep_begin must lie in [0, max_probe_tokens)";
  if (c.defer_v != 0 && c.defer_v != 1) return "defer_v must be 0 or 1";
  if (c.summary_token != 0 && c.summary_token != 1) return "summary_token must be 0 or 1";
  if (c.summary_token && (c.rope_mode != HERMES_ROPE_1D || c.budget < 2))
    return "summary tokens need 1D RoPE (Alg. 1 takes one target index t) and budget >= 2";
  if (c.reindex_mode == HERMES_REINDEX_LAZY) {
    const long long span = c.rope_mode == HERMES_ROPE_M3D
        ? (c.max_chunk_tokens + c.mrope_grid_h * c.mrope_grid_w - 1) / (c.mrope_grid_h * c.mrope_grid_w) : c.max_chunk_tokens;
    if ((long long)c.max_position < (long long)c.pos_offset + c.budget + 2 * span)
      return "lazy re-indexing needs max_position >= pos_offset + budget + 2 chunk spans";
    if (c.max_position > (1 << 20)) return "max_position too large (rotary table)";
  }
  if (c.score_path < HERMES_SCORE_AUTO || c.score_path > HERMES_SCORE_TCGEN05) return "bad score_path";
  for (float w : c.budget_weight) if (!(w > 0.f) || !std::isfinite(w)) return "budget_weight must be positive";
  if (!uniform_budgets(c)) {
    if (c.rope_mode != HERMES_ROPE_1D) return "layer-dependent budgets need 1D RoPE";
    for (int m : layer_budgets(c, ns, nd)) {
      if (m < (c.summary_token ? 2 : 1)) return "a layer's budget would be zero (or, with summary tokens, below 2)";
      if (c.max_tokens != 0 && c.max_tokens <= m) return "max_tokens must exceed the largest layer budget (or be 0)";
    }
  }
  if (size_t(c.budget) + size_t(c.max_chunk_tokens) > (size_t(1) << 24)) return "budget + chunk too large";
  return nullptr;
}

inline Layout make_layout(const hermes_config& c) {
  Layout y{};
  int ns = c.n_shallow, nd = c.n_deep;
  stage_split(c.n_layers, ns, nd);
  y.n_shallow = ns; y.n_deep = nd; y.n_middle = c.n_layers - ns - nd;
  y.budget_max = y.budget_min = c.budget;
  for (int m : layer_budgets(c, ns, nd)) { y.budget_max = std::max(y.budget_max, m); y.budget_min = std::min(y.budget_min, m); }
  y.cap = c.max_tokens ? c.max_tokens : y.budget_max + c.max_chunk_tokens;
  y.n_axes = c.rope_mode == HERMES_ROPE_M3D ? 3 : 1;
  y.esize = c.dtype == HERMES_BF16 ? 2 : 4;
  y.row_bytes = size_t(c.n_kv_heads) * c.head_dim * y.esize;
  y.n_part_max = (y.cap + 127) / 128;
  y.n_vh_max = 4 * c.n_kv_heads * std::max(1, (c.n_q_heads / c.n_kv_heads * c.max_probe_tokens + 511) / 512);
  if (c.rope_mode == HERMES_ROPE_M3D) {
    const int tpt = c.mrope_grid_h * c.mrope_grid_w;
    y.table_rows = c.budget + (c.max_chunk_tokens + tpt - 1) / tpt + 2;
  } else {
    y.table_rows = y.cap - y.budget_min + 1 + (c.summary_token ? 1 : 0);   // summary layers evict one token more
  }
  // lazy mode: a re-index step moves positions from anywhere below the limit down to the compact range
  if (c.reindex_mode == HERMES_REINDEX_LAZY) y.table_rows = std::max(y.table_rows, c.max_position - c.pos_offset + 2);
  const size_t BL = size_t(c.n_streams) * c.n_layers;
  const size_t rows = size_t(c.n_q_heads) * c.max_probe_tokens;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
  y.kc = take(BL * 2 * y.cap * y.row_bytes);
  y.vc = take(BL * 2 * y.cap * y.row_bytes);
  y.posc = take(BL * 2 * y.n_axes * y.cap * 4);
  y.colsum = take(BL * y.n_vh_max * y.cap * 4);
  y.wsum = take(BL * y.cap * 4);
  y.wmax = take(BL * 4);
  y.rowstat = take(BL * rows * 2 * 4);
  y.partial = take(BL * rows * y.n_part_max * 2 * 4);
  y.scores = take(BL * y.cap * 4);
  y.kept = take(BL * y.budget_max * 4);
  y.delta = take(BL * y.n_axes * y.budget_max * 4);
  y.evicted = take(BL * size_t(y.cap - y.budget_min + 1) * 4);
  y.rope_tab = take(size_t(y.table_rows) * (c.head_dim / 2) * 8);
  y.rope_freq = take(size_t(c.head_dim / 2) * 8);
  // summary tokens: (cos, sin)(delta * theta_j) for delta in [-sum_tab_neg, sum_tab_rows - sum_tab_neg).  Eager: an evicted
  // token moves from p in [offset, offset + cap) to t = offset + budget - 1.  Lazy: to the position after the newest token
  // (delta up to max_position - offset), and back down at a re-index step.  Capped at 2 x 65536 rows; beyond: fp64 sincos.
  y.sum_tab_neg = y.cap - y.budget_min + 1;
  int sum_pos = y.budget_max + 1;
  if (c.reindex_mode == HERMES_REINDEX_LAZY) {
    y.sum_tab_neg = std::min(65536, std::max(y.sum_tab_neg, c.max_position - c.pos_offset + 1));
    sum_pos = std::min(65536, std::max(sum_pos, c.max_position - c.pos_offset + 1));
  }
  y.sum_tab_rows = c.summary_token ? y.sum_tab_neg + sum_pos : 0;
  y.sum_tab = take(size_t(y.sum_tab_rows) * (c.head_dim / 2) * 8);
  y.omega = take(size_t(c.n_layers) * 4);
  y.lambda = take(size_t(c.n_layers) * 4);
  y.status = take(256);
  y.seg_cnt = take(BL * y.n_vh_max * 4);
  y.lay_dyn = take(size_t(c.n_layers) * 2 * 4);
  y.tc_pre = take((BL + 1) * 2 * 4);              // layer-dependent budgets on the tcgen05 path: segment / tile prefix sums
  // staging of the host entry point, two sets: the copies of call n + 1 run while the kernels of call n read set n & 1
  y.stage_kv_bytes = align_up(BL * c.max_chunk_tokens * y.row_bytes);
  y.stage_q_bytes = align_up(BL * rows * c.head_dim * y.esize);
  y.stage_k = take(2 * y.stage_kv_bytes);
  y.stage_v = take(2 * y.stage_kv_bytes);
  y.stage_q = take(2 * y.stage_q_bytes);
  y.tmaps = take(4096);
  y.total = o;
  return y;
}

// Launch with programmatic stream serialization allowed (see pdl_wait() in common.cuh).
template <typename... P, typename... A>
inline cudaError_t launch_pdl(void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, A... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, P(args)...);
}

// Same, as a COOPERATIVE launch: the runtime refuses the launch (cudaErrorCooperativeLaunchTooLarge) unless every CTA of the
// grid can be resident at once -- which is what a kernel whose CTAs wait on one another needs.
template <typename... P, typename... A>
inline cudaError_t launch_pdl_coop(void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, A... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  at[1].id = cudaLaunchAttributeCooperative;
  at[1].val.cooperative = 1;
  cfg.attrs = at; cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, kernel, P(args)...);
}

struct KernelTimer {
  cudaEvent_t beg[HERMES_K_COUNT]{}, end[HERMES_K_COUNT]{};
  bool ran[HERMES_K_COUNT]{};
  bool created = false;
};

}  // namespace hk

struct hermes {
  hermes_config cfg{};
  hk::Layout lay{};
  hk::Geom geom{};
  char* ws = nullptr;
  int len = 0;              // tokens per layer (host-tracked; identical for all streams / layers; LB: the largest layer's)
  bool lb = false;          // layer-dependent budgets (DESIGN f4)
  std::vector<int> lay_budget, lay_len, lay_last_T;   // per layer: m_l, tokens held, candidates at the last eviction
  int cur = 0;              // which half of the double buffer is current
  long long t_steps_seen = 0;   // M-RoPE temporal steps appended so far
  long long next_pos = 0;   // smallest admissible pos_start of the next chunk
  int last_T = 0;
  int last_score_path = 0;
  int last_launches = 0;
  int n_sm = 148;
  // host entry point: all host-to-device copies run on a library-owned copy stream (created on first use), into
  // staging set (call count & 1); ev_free[p] = the kernels that read set p have been enqueued and executed
  cudaStream_t side_stream = nullptr;
  cudaEvent_t ev_k_done[2] = {nullptr, nullptr}, ev_v_done[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
  bool ev_free_set[2] = {false, false};
  unsigned host_calls = 0;
  int n_vh = 0;             // column-sum slots written by the last scoring pass
  // deferred V compaction: after an eviction on the tcgen05 path k_gather moves only K; the kept V rows still sit
  // in buffer v_src_buf and are moved into the current buffer by the NEXT update's scoring kernel (or by a flush)
  bool v_pending = false;
  int v_src_buf = 0;
  void* last_stream = nullptr;
  bool profiling = false;
  bool tc_ok = false;       // tcgen05 scoring path usable for this config + device
  hk::KernelTimer timer;
  std::string err;
  void* tc_state = nullptr; // opaque state of the tensor-core scoring path (tensor maps, ...)
};
