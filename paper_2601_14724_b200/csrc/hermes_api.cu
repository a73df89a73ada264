// C-ABI entry points (include/hermes.h): config validation, workspace carve-up, and the stream-ordered
// launch sequence of one chunk arrival.  No host synchronisation on the success path of an append.
#include <climits>

#include "host_state.cuh"
#include "k_append.cuh"
#include "k_gather.cuh"
#include "k_score_simt.cuh"
#include "k_select.cuh"
#include "k_summary.cuh"
#include "k_score_tc.cuh"

using namespace hk;

static thread_local std::string g_create_error;

namespace {
template <typename T> struct TypeTag { using type = T; };
void flush_v(hermes_t* h, cudaStream_t s);   // runs a deferred V compaction on its own
}  // namespace

static int fail(hermes_t* h, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (h) h->err = buf; else g_create_error = buf;
  return code;
}

#define CUDA_TRY(h, call)                                                                     \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) return fail(h, HERMES_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

extern "C" void hermes_default_config(hermes_config* c) {
  if (!c) return;
  memset(c, 0, sizeof *c);
  c->n_streams = 1;
  c->dtype = HERMES_BF16;
  c->n_shallow = c->n_deep = c->l_short = c->l_long = -1;
  c->omega0 = 0.75f; c->gamma = 0.6f;
  c->lambda_shallow = 0.1f; c->lambda_middle = 0.3f; c->lambda_deep = 0.4f;
  c->norm_mode = HERMES_NORM_MAX;
  c->rope_mode = HERMES_ROPE_1D; c->rope_theta = 10000.f;
  c->mrope_section[0] = 16; c->mrope_section[1] = 24; c->mrope_section[2] = 24;
  c->mrope_compact_axes = 1; c->mrope_grid_h = 8; c->mrope_grid_w = 8;
  c->max_probe_tokens = 64;
  c->score_path = HERMES_SCORE_AUTO;
  c->reindex_mode = HERMES_REINDEX_EAGER;
  c->defer_v = 1;
  c->budget_weight[0] = c->budget_weight[1] = c->budget_weight[2] = 1.f;
}

extern "C" size_t hermes_workspace_bytes(const hermes_config* c) {
  if (!c || validate(*c)) return 0;
  return make_layout(*c).total;
}

extern "C" int hermes_layer_budgets(const hermes_config* c, int32_t* out, int32_t n) {
  if (!c || !out || n < 0) return HERMES_EINVAL;
  if (const char* why = validate(*c)) { g_create_error = why; return HERMES_EINVAL; }
  int ns = c->n_shallow, nd = c->n_deep;
  stage_split(c->n_layers, ns, nd);
  const std::vector<int> m = layer_budgets(*c, ns, nd);
  for (int l = 0; l < c->n_layers && l < n; ++l) out[l] = m[l];
  return c->n_layers;
}

extern "C" const char* hermes_last_error(const hermes_t* h) { return h ? h->err.c_str() : g_create_error.c_str(); }
extern "C" int32_t hermes_len(const hermes_t* h) { return h ? h->len : 0; }
extern "C" int32_t hermes_layer_len(const hermes_t* h, int32_t layer) {
  if (!h || layer < 0 || layer >= h->cfg.n_layers) return -1;
  return h->lb ? h->lay_len[layer] : h->len;
}
extern "C" int32_t hermes_layer_budget(const hermes_t* h, int32_t layer) {
  if (!h || layer < 0 || layer >= h->cfg.n_layers) return -1;
  return h->lay_budget[layer];
}
extern "C" int32_t hermes_last_score_path(const hermes_t* h) { return h ? h->last_score_path : 0; }
extern "C" int32_t hermes_v_pending(const hermes_t* h) { return h && h->v_pending ? 1 : 0; }
extern "C" int32_t hermes_last_launch_count(const hermes_t* h) { return h ? h->last_launches : 0; }

extern "C" int hermes_create(const hermes_config* c, void* workspace, size_t bytes, hermes_t** out) {
  if (out) *out = nullptr;
  if (!c || !out) return fail(nullptr, HERMES_EINVAL, "null argument");
  if (const char* why = validate(*c)) return fail(nullptr, HERMES_EINVAL, "%s", why);
  const Layout y = make_layout(*c);
  if (!workspace) return fail(nullptr, HERMES_EINVAL, "null workspace");
  if (reinterpret_cast<uintptr_t>(workspace) % 256) return fail(nullptr, HERMES_EINVAL, "workspace must be 256-byte aligned");
  if (bytes < y.total) return fail(nullptr, HERMES_ECAPACITY, "workspace of %zu bytes < %zu needed", bytes, y.total);

  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0 || c->device < 0 || c->device >= n_dev) {
    (void)cudaGetLastError();
    return fail(nullptr, HERMES_ECUDA, "no usable CUDA device %d (found %d): this library has no CPU fallback", c->device, n_dev);
  }
  cudaDeviceProp prop;
  CUDA_TRY(nullptr, cudaGetDeviceProperties(&prop, c->device));
  if (prop.major != 10) return fail(nullptr, HERMES_ECUDA, "device %d is sm_%d%d; kernels are built for sm_100a only", c->device, prop.major, prop.minor);
  CUDA_TRY(nullptr, cudaSetDevice(c->device));
  {
    cudaFuncAttributes fa;
    CUDA_TRY(nullptr, cudaFuncGetAttributes(&fa, k_select));
    if (fa.sharedSizeBytes + size_t(y.cap) * 4 > prop.sharedMemPerBlockOptin)
      return fail(nullptr, HERMES_EINVAL, "max_tokens %d too large for the select kernel's shared memory", y.cap);
    if (c->summary_token) {
      const size_t need = size_t(y.cap - y.budget_min + 2) * 8;
      cudaFuncAttributes fs;
      CUDA_TRY(nullptr, c->dtype == HERMES_BF16 ? cudaFuncGetAttributes(&fs, k_summary<__nv_bfloat16>) : cudaFuncGetAttributes(&fs, k_summary<float>));
      if (fs.sharedSizeBytes + need > prop.sharedMemPerBlockOptin)
        return fail(nullptr, HERMES_EINVAL, "max_chunk_tokens %d too large for the summary kernel's shared memory", c->max_chunk_tokens);
      CUDA_TRY(nullptr, c->dtype == HERMES_BF16
                            ? cudaFuncSetAttribute(k_summary<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(need))
                            : cudaFuncSetAttribute(k_summary<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(need)));
    }
  }
  const int n_sm = prop.multiProcessorCount;

  hermes_t* h = new (std::nothrow) hermes;
  if (!h) return fail(nullptr, HERMES_ENOMEM, "out of host memory");
  h->cfg = *c; h->lay = y; h->ws = static_cast<char*>(workspace);
  h->next_pos = c->pos_offset;
  h->n_sm = n_sm;

  Geom& g = h->geom;
  g.B = c->n_streams; g.L = c->n_layers; g.Hq = c->n_q_heads; g.Hkv = c->n_kv_heads;
  g.G = c->n_q_heads / c->n_kv_heads; g.d = c->head_dim;
  // layer-dependent budgets: g.budget is the stride of the kept / delta lists (the largest layer budget); the per-layer
  // counts come from lay_T / lay_keep, rewritten before every update
  h->lb = !uniform_budgets(*c);
  h->lay_budget = layer_budgets(*c, y.n_shallow, y.n_deep);
  h->lay_len.assign(c->n_layers, 0); h->lay_last_T.assign(c->n_layers, 0);
  g.cap = y.cap; g.budget = y.budget_max; g.n_axes = y.n_axes; g.row_elems = c->n_kv_heads * c->head_dim;
  g.lay_T = h->lb ? reinterpret_cast<const int32_t*>(h->ws + y.lay_dyn) : nullptr;
  g.lay_keep = h->lb ? g.lay_T + c->n_layers : nullptr;
  g.n_shallow = y.n_shallow; g.n_deep = y.n_deep; g.summary = c->summary_token; g.probe_deep_begin = c->probe_deep_begin; g.n_evict_max = y.cap - y.budget_min + 1;
  g.p_max = c->max_probe_tokens; g.pos_offset = c->pos_offset;
  g.sec_t = c->mrope_section[0]; g.sec_h = c->mrope_section[1];
  g.compact_axes = c->mrope_compact_axes; g.grid_h = c->mrope_grid_h; g.grid_w = c->mrope_grid_w;
  g.table_rows = y.table_rows; g.n_vh_max = y.n_vh_max;
  g.kc = h->ws + y.kc; g.vc = h->ws + y.vc; g.posc = reinterpret_cast<int32_t*>(h->ws + y.posc);
  g.colsum = reinterpret_cast<float*>(h->ws + y.colsum);
  g.rowstat = reinterpret_cast<float*>(h->ws + y.rowstat);
  g.wsum = reinterpret_cast<float*>(h->ws + y.wsum);
  g.wmax = reinterpret_cast<uint32_t*>(h->ws + y.wmax);
  g.partial = reinterpret_cast<float*>(h->ws + y.partial);
  g.scores = reinterpret_cast<float*>(h->ws + y.scores);
  g.kept = reinterpret_cast<int32_t*>(h->ws + y.kept);
  g.delta = reinterpret_cast<int32_t*>(h->ws + y.delta);
  g.evicted = reinterpret_cast<int32_t*>(h->ws + y.evicted);
  g.rope_tab = reinterpret_cast<float2*>(h->ws + y.rope_tab);
  g.rope_freq = reinterpret_cast<double*>(h->ws + y.rope_freq);
  g.sum_tab = reinterpret_cast<float2*>(h->ws + y.sum_tab);
  g.sum_tab_zero = y.sum_tab_neg; g.sum_tab_rows = y.sum_tab_rows;
  g.omega = reinterpret_cast<float*>(h->ws + y.omega);
  g.lambda = reinterpret_cast<float*>(h->ws + y.lambda);
  g.status = reinterpret_cast<int32_t*>(h->ws + y.status);
  g.seg_cnt = reinterpret_cast<unsigned*>(h->ws + y.seg_cnt);

  // per-layer recency weight (Eq. 3-4) and smoothing weight (Eq. 7)
  const int L = c->n_layers, ns = y.n_shallow, nm = y.n_middle;
  const int l_short = c->l_short >= 0 ? c->l_short : ns;
  const int l_long = c->l_long >= 0 ? c->l_long : ns + nm - 1;
  std::vector<float> omega(L), lambda(L);
  for (int l = 0; l < L; ++l) {
    if (l < ns) { omega[l] = 1.f; lambda[l] = c->lambda_shallow; }
    else if (l < ns + nm) {
      omega[l] = l_long == l_short ? c->omega0
                                   : float(double(c->omega0) - double(c->gamma) * double(l - l_short) / double(l_long - l_short));
      lambda[l] = c->lambda_middle;
    } else { omega[l] = 0.f; lambda[l] = c->lambda_deep; }
  }
  // rotary angle table in fp64: row r holds (cos, sin)(delta * theta_j) for delta = -r
  const int half = c->head_dim / 2;
  std::vector<double> freq(half);
  for (int j = 0; j < half; ++j) freq[j] = std::pow(double(c->rope_theta), -2.0 * double(j) / double(c->head_dim));
  std::vector<float2> tab(size_t(y.table_rows) * half);
  for (int r = 0; r < y.table_rows; ++r)
    for (int j = 0; j < half; ++j) {
      const double ang = double(-r) * freq[j];
      tab[size_t(r) * half + j] = make_float2(float(std::cos(ang)), float(std::sin(ang)));
    }
  cudaError_t e = cudaSuccess;
  auto up = [&](void* dst, const void* src, size_t n) { if (e == cudaSuccess) e = cudaMemcpy(dst, src, n, cudaMemcpyHostToDevice); };
  up(g.omega, omega.data(), L * 4); up(g.lambda, lambda.data(), L * 4);
  up(g.rope_freq, freq.data(), half * 8); up(g.rope_tab, tab.data(), tab.size() * 8);

  if (c->summary_token) {                          // (cos, sin)(delta * theta_j) for every delta Alg. 1 can meet
    std::vector<float2> st(size_t(y.sum_tab_rows) * half);
    for (int r = 0; r < y.sum_tab_rows; ++r)
      for (int j = 0; j < half; ++j) {
        const double ang = double(r - g.sum_tab_zero) * freq[j];
        st[size_t(r) * half + j] = make_float2(float(std::cos(ang)), float(std::sin(ang)));
      }
    up(g.sum_tab, st.data(), st.size() * 8);
  }
  if (e == cudaSuccess) e = cudaMemset(g.status, 0, 256);
  if (e == cudaSuccess) e = cudaMemset(h->ws + y.seg_cnt, 0, size_t(g.B) * L * y.n_vh_max * 4);
  if (e == cudaSuccess) e = cudaMemset(g.posc, 0, size_t(g.B) * L * 2 * y.n_axes * y.cap * 4);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_select, cudaFuncAttributeMaxDynamicSharedMemorySize, y.cap * 4);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  if (e != cudaSuccess) {
    fail(nullptr, HERMES_ECUDA, "create: %s", cudaGetErrorString(e));
    delete h;
    return HERMES_ECUDA;
  }
  // tensor-core scoring path: bf16, d = 128; probing it builds its tensor maps
  h->tc_ok = tc_init(h);
  if (c->score_path == HERMES_SCORE_TCGEN05 && !h->tc_ok) {
    std::string why = h->err;
    delete h;
    return fail(nullptr, HERMES_EINVAL, "tcgen05 scoring path unavailable for this config: %s", why.c_str());
  }
  *out = h;
  return HERMES_OK;
}

extern "C" void hermes_destroy(hermes_t* h) {
  if (!h) return;
  if (h->timer.created)
    for (int i = 0; i < HERMES_K_COUNT; ++i) { cudaEventDestroy(h->timer.beg[i]); cudaEventDestroy(h->timer.end[i]); }
  if (h->side_stream) {
    cudaStreamSynchronize(h->side_stream); cudaStreamDestroy(h->side_stream);
    for (int p = 0; p < 2; ++p) { cudaEventDestroy(h->ev_k_done[p]); cudaEventDestroy(h->ev_v_done[p]); cudaEventDestroy(h->ev_free[p]); }
  }
  tc_destroy(h);
  delete h;
}

extern "C" int hermes_set_profiling(hermes_t* h, int32_t enable) {
  if (!h) return HERMES_EINVAL;
  if (enable && !h->timer.created) {
    for (int i = 0; i < HERMES_K_COUNT; ++i) {
      CUDA_TRY(h, cudaEventCreate(&h->timer.beg[i]));
      CUDA_TRY(h, cudaEventCreate(&h->timer.end[i]));
    }
    h->timer.created = true;
  }
  h->profiling = enable != 0;
  return HERMES_OK;
}

extern "C" int hermes_get_profile(hermes_t* h, float* ms_out, int32_t n) {
  if (!h || !ms_out || n < 0) return HERMES_EINVAL;
  if (!h->timer.created) return fail(h, HERMES_ESTATE, "profiling was never enabled");
  int w = 0;
  for (; w < n && w < HERMES_K_COUNT; ++w) {
    ms_out[w] = 0.f;
    if (!h->timer.ran[w]) continue;
    CUDA_TRY(h, cudaEventSynchronize(h->timer.end[w]));
    CUDA_TRY(h, cudaEventElapsedTime(&ms_out[w], h->timer.beg[w], h->timer.end[w]));
  }
  return w;
}

extern "C" int hermes_device_status(hermes_t* h, int32_t* status_out) {
  if (!h || !status_out) return HERMES_EINVAL;
  CUDA_TRY(h, cudaMemcpy(status_out, h->geom.status, 4, cudaMemcpyDeviceToHost));
  return HERMES_OK;
}

extern "C" int hermes_get_cache(hermes_t* h, int32_t stream, int32_t layer, hermes_cache_view* out) {
  if (!h || !out) return HERMES_EINVAL;
  if (stream < 0 || stream >= h->cfg.n_streams || layer < 0 || layer >= h->cfg.n_layers)
    return fail(h, HERMES_EINVAL, "stream %d / layer %d out of range", stream, layer);
  const Geom& g = h->geom;
  if (h->v_pending) {                       // make V whole before handing out pointers (stream of the last append)
    flush_v(h, static_cast<cudaStream_t>(h->last_stream));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, HERMES_ECUDA, "V compaction: %s", cudaGetErrorString(e));
  }
  const size_t bl = size_t(stream) * g.L + layer, slab = bl * 2 + h->cur;
  out->k = static_cast<char*>(g.kc) + slab * g.cap * h->lay.row_bytes;
  out->v = static_cast<char*>(g.vc) + slab * g.cap * h->lay.row_bytes;
  out->pos = g.posc + slab * g.n_axes * g.cap;
  out->n_axes = g.n_axes; out->pos_stride = g.cap; out->len = h->lb ? h->lay_len[layer] : h->len;
  out->last_T = h->lb ? h->lay_last_T[layer] : h->last_T;
  out->last_scores = h->last_T ? g.scores + bl * g.cap : nullptr;
  out->last_kept = h->last_T ? g.kept + bl * g.budget : nullptr;
  return HERMES_OK;
}

namespace {
struct Prof {                               // brackets one kernel with events when profiling is on
  hermes_t* h; int id; cudaStream_t s;
  Prof(hermes_t* h_, int id_, cudaStream_t s_) : h(h_), id(id_), s(s_) {
    if (h->profiling) { cudaEventRecord(h->timer.beg[id], s); h->timer.ran[id] = true; }
    ++h->last_launches;
  }
  ~Prof() { if (h->profiling) cudaEventRecord(h->timer.end[id], s); }
};

template <typename T>
void launch_simt(hermes_t* h, const void* q, int Tn, int P, float scale_log2, cudaStream_t s) {
  const Geom& g = h->geom;
  const int n_part = (Tn + kSimtTokens - 1) / kSimtTokens;
  const dim3 grid(n_part, g.Hkv, g.B * (g.L - g.n_shallow));
  const T* qp = static_cast<const T*>(q);
  auto run = [&](auto dconst) {
    constexpr int D = decltype(dconst)::value;
    { Prof p(h, HERMES_K_SCORE_STATS, s);
      k_score_simt<T, D, false><<<grid, kSimtTokens, 0, s>>>(g, qp, h->cur, Tn, P, scale_log2, n_part); }
    { Prof p(h, HERMES_K_SCORE_COMBINE, s);
      const int warps = g.B * (g.L - g.n_shallow) * g.Hq * P;
      k_score_combine<<<(warps + 7) / 8, 256, 0, s>>>(g, P, n_part); }
    { Prof p(h, HERMES_K_SCORE_COLSUM, s);
      k_score_simt<T, D, true><<<grid, kSimtTokens, 0, s>>>(g, qp, h->cur, Tn, P, scale_log2, n_part); }
  };
  if (g.d == 32) run(std::integral_constant<int, 32>{});
  else if (g.d == 64) run(std::integral_constant<int, 64>{});
  else run(std::integral_constant<int, 128>{});
}
// k_gather for buffer `buf` -> buf ^ 1 in the given mode (kGatherKV / kGatherK / kGatherV).
void launch_gather(hermes_t* h, int mode, int buf, cudaStream_t s) {
  const hermes_config& c = h->cfg;
  const Geom& g = h->geom;
  const int BL = g.B * g.L;
  ++h->last_launches;
  const int V = c.dtype == HERMES_BF16 ? 8 : 4;
  const int upr = g.Hkv * (g.d / 2 / V);
  const int total = g.budget * upr;
  // 4 resident blocks per SM, whole waves only (a partial extra wave, as the old rounding produced, cost 5 us);
  // K + V launches: 8 waves measured best (118 -> 114 us at configs[1]: short blocks even out the per-SM HBM rates)
  const int waves = mode == kGatherK ? 2 : 8;     // the K-only launch prefers long blocks: 69.6 us at 2 waves, 72.2 at 8, 81 at 24
  const int per_wave = h->n_sm * 4;
  const int gx_max = std::max(1, (total + kGatherThreads - 1) / kGatherThreads);
  int gx = std::max(1, std::min((per_wave * waves) / BL, gx_max));
  // many slabs (batched streams): gridDim.x would round down to 1-2 and leave the last wave mostly empty -- take the
  // smallest blocks-per-slab count that fills whole waves best (configs[4], 640 slabs: K gather 5.1 -> 4.1 ms)
  if (BL > per_wave * waves / 2) {
    double best = 0.0;
    for (int cand = 1; cand <= std::min(16, gx_max); ++cand) {
      const double w = double(cand) * BL / per_wave, fill = w / std::ceil(w);
      if (fill > best + 1e-9) { best = fill; gx = cand; }
    }
  }
  const dim3 grid(gx, BL), block(kGatherThreads);
  auto go = [&](auto tag, auto nax, auto md) {
    using T = typename decltype(tag)::type;
    launch_pdl(k_gather<T, decltype(nax)::value, decltype(md)::value>, grid, block, 0, s, g, buf);
  };
  auto by_mode = [&](auto tag, auto nax) {
    if (mode == kGatherKV) go(tag, nax, std::integral_constant<int, kGatherKV>{});
    else if (mode == kGatherK) go(tag, nax, std::integral_constant<int, kGatherK>{});
    else go(tag, nax, std::integral_constant<int, kGatherV>{});
  };
  auto by_axes = [&](auto tag) {
    if (g.n_axes == 1) by_mode(tag, std::integral_constant<int, 1>{});
    else by_mode(tag, std::integral_constant<int, 3>{});
  };
  if (c.dtype == HERMES_BF16) by_axes(TypeTag<__nv_bfloat16>{});
  else by_axes(TypeTag<float>{});
}

// Runs a deferred V compaction on its own (no scoring kernel to carry it).
void flush_v(hermes_t* h, cudaStream_t s) {
  if (!h->v_pending) return;
  launch_gather(h, kGatherV, h->v_src_buf, s);
  h->v_pending = false;
}
}  // namespace

// v_ready != NULL (host entry point): V_new is still being copied on another stream; its rows are appended by a second
// k_append launch once the scoring kernels are enqueued, behind a wait on that event.
static int append_impl(hermes_t* h, const void* K_new, const void* V_new, const void* Q_probe,
                       int32_t n_new, int32_t n_probe, int32_t pos_start, void* cuda_stream, cudaEvent_t v_ready) {
  if (!h) return HERMES_EINVAL;
  const hermes_config& c = h->cfg;
  Geom& g = h->geom;
  if (!K_new || !V_new) return fail(h, HERMES_EINVAL, "K_new / V_new must not be NULL");
  if (n_new <= 0) return fail(h, HERMES_EINVAL, "n_new = %d must be positive", n_new);
  if (Q_probe && (n_probe <= 0 || n_probe > c.max_probe_tokens)) return fail(h, HERMES_EINVAL, "n_probe = %d not in [1, %d]", n_probe, c.max_probe_tokens);
  if (Q_probe && c.probe_deep_begin >= n_probe) return fail(h, HERMES_EINVAL, "probe_deep_begin %d leaves no probe row of %d for the deep layers", c.probe_deep_begin, n_probe);
  const int Tn = h->len + n_new;                  // layer-dependent budgets: the largest layer's candidates
  if (Tn > g.cap) return fail(h, HERMES_ECAPACITY, "len %d + n_new %d exceeds max_tokens %d", h->len, n_new, g.cap);
  // arrival positions (DESIGN c16): host-computable, strictly above every cached position
  long long p0;
  long long steps = 0;
  const bool lazy = c.reindex_mode == HERMES_REINDEX_LAZY;
  long long span = n_new;                       // positions the chunk spans on the re-indexed axis
  if (g.n_axes == 1) {
    p0 = pos_start >= 0 ? pos_start : (lazy ? h->next_pos : c.pos_offset + h->len);
  } else {
    const int tpt = c.mrope_grid_h * c.mrope_grid_w;
    steps = (n_new + tpt - 1) / tpt;
    span = steps;
    p0 = pos_start >= 0 ? pos_start : (lazy ? h->next_pos : c.pos_offset + std::min<long long>(h->t_steps_seen, c.budget));
  }
  if (p0 < h->next_pos) return fail(h, HERMES_EINVAL, "pos_start %lld is not above the cached positions (need >= %lld)", p0, h->next_pos);
  if (p0 + std::max<long long>(n_new, steps) >= INT_MAX) return fail(h, HERMES_EINVAL, "position overflow");
  bool evict = Q_probe != nullptr && Tn > c.budget;
  std::vector<int32_t> dyn;                       // layer-dependent budgets: [T_l | tokens held after this update]
  if (h->lb) {
    dyn.resize(2 * size_t(c.n_layers));
    evict = false;
    for (int l = 0; l < c.n_layers; ++l) {
      const int T_l = h->lay_len[l] + n_new;
      const bool over = Q_probe != nullptr && T_l > h->lay_budget[l];   // a layer compresses when IT exceeds its budget
      dyn[l] = T_l; dyn[c.n_layers + l] = over ? h->lay_budget[l] : T_l;
      evict |= over;
    }
  }
  // the lazy re-index trigger reasons about "the next chunk" with max_chunk_tokens; elsewhere only the capacity binds
  if (lazy && evict && n_new > c.max_chunk_tokens)
    return fail(h, HERMES_EINVAL, "n_new = %d exceeds max_chunk_tokens %d (lazy re-indexing)", n_new, c.max_chunk_tokens);
  // lazy mode: re-index only when the next chunk would no longer fit below max_position
  const long long span_max = g.n_axes == 1 ? c.max_chunk_tokens
                                           : (c.max_chunk_tokens + c.mrope_grid_h * c.mrope_grid_w - 1) / (c.mrope_grid_h * c.mrope_grid_w);
  // a summary token takes the position after the newest token (DESIGN f1): the running counter advances by one more
  int summ_pos = (c.summary_token && h->lay.n_deep > 0) ? 1 : 0;
  int n_ev_max = Tn - c.budget + 1;                  // longest evicted list a summary token is made of
  if (h->lb && summ_pos) {                           // layer-dependent budgets: only if a deep layer compresses at this arrival
    summ_pos = 0; n_ev_max = 0;
    for (int l = c.n_layers - h->lay.n_deep; l < c.n_layers; ++l)
      if (dyn[c.n_layers + l] < dyn[l]) { summ_pos = 1; n_ev_max = std::max(n_ev_max, int(dyn[l] - dyn[c.n_layers + l] + 1)); }
  }
  const bool reindex = !lazy || p0 + span + summ_pos + span_max > c.max_position;
  if (lazy && p0 + span > c.max_position) return fail(h, HERMES_ECAPACITY, "positions would exceed max_position %d", c.max_position);

  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  h->last_launches = 0;
  for (bool& r : h->timer.ran) r = false;
  const int row_vecs = int(h->lay.row_bytes / 16);
  const int BL = g.B * g.L;
  // tokens the scoring launch spans: with layer-dependent budgets the largest SCORED layer's candidates (k_tc_score<true>
  // masks the rest per layer); shallow layers, which may hold more, are not scored
  int Tn_sc = Tn;
  if (h->lb) { Tn_sc = 1; for (int l = g.n_shallow; l < c.n_layers; ++l) Tn_sc = std::max(Tn_sc, int(dyn[l])); }
  const bool use_tc = evict && g.L > g.n_shallow && h->tc_ok && c.score_path != HERMES_SCORE_SIMT &&
                      (c.score_path == HERMES_SCORE_TCGEN05 || tc_profitable(h, Tn_sc, n_probe));
  h->last_stream = cuda_stream;
  // a pending V compaction rides in this update's scoring kernel if that kernel is long enough and has the
  // shared memory for it; otherwise it runs on its own first
  const bool ride = use_tc && tc_v_ride_ok(h, Tn_sc, n_probe);
  if (!ride) flush_v(h, s);
  // the per-layer tables of THIS update, stream-ordered behind the previous update's kernels and behind a flush (which reads
  // the previous update's counts); the source is pageable memory, so the call has staged it on return
  if (h->lb) CUDA_TRY(h, cudaMemcpyAsync(h->ws + h->lay.lay_dyn, dyn.data(), dyn.size() * 4, cudaMemcpyHostToDevice, s));
  {
    Prof p(h, HERMES_K_APPEND, s);
    const size_t n_vec = size_t(n_new) * row_vecs;
    const int gx = int(std::min<size_t>((n_vec + 511) / 512, 64));
    launch_pdl(k_append, dim3(std::max(gx, 1), BL), dim3(256), 0, s, g, static_cast<const uint4*>(K_new), static_cast<const uint4*>(V_new),
               h->cur, h->len, n_new, row_vecs, int(p0), v_ready ? kAppendK : (kAppendK | kAppendV));
  }
  auto append_v_late = [&]() {                       // nothing before the gather (or a later reader) needs V_new
    if (!v_ready) return;
    cudaStreamWaitEvent(s, v_ready, 0);
    const size_t n_vec = size_t(n_new) * row_vecs;
    const int gx = int(std::min<size_t>((n_vec + 511) / 512, 64));
    launch_pdl(k_append, dim3(std::max(gx, 1), BL), dim3(256), 0, s, g, static_cast<const uint4*>(K_new), static_cast<const uint4*>(V_new),
               h->cur, h->len, n_new, row_vecs, int(p0), kAppendV);
    ++h->last_launches;
  };
  if (!evict) append_v_late();
  if (evict) {
    const float scale = c.softmax_scale > 0.f ? c.softmax_scale : float(1.0 / std::sqrt(double(c.head_dim)));
    const float scale_log2 = scale * kLog2e;
    if (g.L > g.n_shallow) {
      bool scored = false;
      if (use_tc) {
        const int rc = tc_score(h, Q_probe, Tn_sc, n_new, n_probe, scale_log2, s, ride && h->v_pending);
        if (rc == kTcNotResident) {
          // the device cannot hold one scoring CTA per unit of its grid at once (MPS / green-context partition): this
          // handle scores on the CUDA-core path from now on; a pending V compaction runs on its own
          if (c.score_path == HERMES_SCORE_TCGEN05) return fail(h, HERMES_ECUDA, "tcgen05 scoring kernel cannot be made resident on this device partition");
          h->tc_ok = false;
          if (h->lb && h->v_pending) {               // the flush counts rows with the PREVIOUS update's table: put it back for it
            std::vector<int32_t> prev(dyn);
            for (int l = 0; l < c.n_layers; ++l) prev[c.n_layers + l] = h->lay_len[l];
            CUDA_TRY(h, cudaMemcpyAsync(h->ws + h->lay.lay_dyn, prev.data(), prev.size() * 4, cudaMemcpyHostToDevice, s));
            flush_v(h, s);
            CUDA_TRY(h, cudaMemcpyAsync(h->ws + h->lay.lay_dyn, dyn.data(), dyn.size() * 4, cudaMemcpyHostToDevice, s));
          } else {
            flush_v(h, s);
          }
        } else if (rc != HERMES_OK) {
          return rc;
        } else {
          h->v_pending = false;
          h->last_score_path = HERMES_SCORE_TCGEN05;
          scored = true;
        }
      }
      if (!scored) {
        if (c.dtype == HERMES_BF16) launch_simt<__nv_bfloat16>(h, Q_probe, Tn, n_probe, scale_log2, s);
        else launch_simt<float>(h, Q_probe, Tn, n_probe, scale_log2, s);
        h->last_score_path = HERMES_SCORE_SIMT;
        h->n_vh = g.Hkv;
      }
    }
    append_v_late();
    {
      Prof p(h, HERMES_K_SELECT, s);
      if (g.L > g.n_shallow) ++h->last_launches;
      const double k = c.forget_rate;
      const float r_norm_sum = float((1.0 - std::exp(-k)) / (1.0 - std::exp(-k * Tn)));
      if (g.L > g.n_shallow)
        launch_pdl(k_wsum, dim3((Tn + 255) / 256, g.B * (g.L - g.n_shallow)), dim3(256), 0, s, g, Tn, n_probe, h->n_vh);
      launch_pdl(k_select, dim3(BL), dim3(kSelThreads), size_t(Tn) * 4, s, g, h->cur, Tn, c.forget_rate, int(c.norm_mode == HERMES_NORM_SUM), r_norm_sum, int(reindex),
                 reindex ? c.pos_offset + c.budget - 1 : int(p0 + span));
    }
    if (summ_pos) {
      Prof p(h, HERMES_K_SUMMARY, s);
      const dim3 sgrid(g.Hkv, g.B * h->lay.n_deep), sblock(64 * kSumLanes);
      const size_t ssm = size_t(n_ev_max) * 8;
      const int st_pos = int(p0 + span);                 // target between re-index steps; at one: offset + m_l - 1, per layer
      const cudaError_t es = c.dtype == HERMES_BF16 ? launch_pdl(k_summary<__nv_bfloat16>, sgrid, sblock, ssm, s, g, h->cur, Tn, st_pos, int(reindex))
                                                    : launch_pdl(k_summary<float>, sgrid, sblock, ssm, s, g, h->cur, Tn, st_pos, int(reindex));
      if (es != cudaSuccess) return fail(h, HERMES_ECUDA, "summary kernel launch: %s", cudaGetErrorString(es));
    }
    {
      if (h->profiling) { cudaEventRecord(h->timer.beg[HERMES_K_GATHER], s); h->timer.ran[HERMES_K_GATHER] = true; }
      // on the tcgen05 path V stays behind: the next update's scoring kernel compacts it (tc_v_mover), or a flush
      const bool defer_v = ride && c.defer_v != 0;   // the next update will most likely look like this one
      launch_gather(h, defer_v ? kGatherK : kGatherKV, h->cur, s);
      if (defer_v) { h->v_pending = true; h->v_src_buf = h->cur; }
      if (h->profiling) cudaEventRecord(h->timer.end[HERMES_K_GATHER], s);
    }
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, HERMES_ECUDA, "kernel launch failed: %s", cudaGetErrorString(e));
  // commit host-tracked state
  if (g.n_axes == 3) h->t_steps_seen += steps;
  if (h->lb) {
    int mx = 0;
    bool untouched = false;                         // a layer under its budget keeps its original positions
    for (int l = 0; l < c.n_layers; ++l) {
      if (evict) h->lay_last_T[l] = dyn[l];
      h->lay_len[l] = evict ? dyn[c.n_layers + l] : dyn[l];
      untouched |= dyn[c.n_layers + l] == dyn[l];
      mx = std::max(mx, h->lay_len[l]);
    }
    if (evict) { h->cur ^= 1; h->last_T = Tn; }
    h->len = mx;
    // after a re-index step every position of a layer that compressed is below offset + m_l (DESIGN f4)
    h->next_pos = (!evict || !reindex) ? p0 + n_new + (evict ? summ_pos : 0) : std::max<long long>(c.pos_offset + mx, untouched ? p0 + n_new : 0);
  } else if (evict) {
    h->cur ^= 1; h->len = c.budget; h->last_T = Tn;
    if (!reindex) h->next_pos = p0 + span + summ_pos; else
    // after eager re-indexing every cached position is below offset + budget (1D) or below
    // offset + min(temporal steps seen, budget) (M-RoPE: a layer holds at most that many distinct t)
    h->next_pos = c.pos_offset + (g.n_axes == 1 ? (long long)c.budget : std::min<long long>(h->t_steps_seen, c.budget));
  } else {
    h->len = Tn;
    h->next_pos = p0 + (g.n_axes == 1 ? n_new : steps);
  }
  return HERMES_OK;
}

extern "C" int hermes_append_chunk(hermes_t* h, const void* K_new, const void* V_new, const void* Q_probe,
                                   int32_t n_new, int32_t n_probe, int32_t pos_start, void* cuda_stream) {
  return append_impl(h, K_new, V_new, Q_probe, n_new, n_probe, pos_start, cuda_stream, nullptr);
}

extern "C" int hermes_append_chunk_host(hermes_t* h, const void* K_host, const void* V_host, const void* Q_host,
                                        int32_t n_new, int32_t n_probe, int32_t pos_start,
                                        int32_t* kept_out_host, void* cuda_stream) {
  if (!h) return HERMES_EINVAL;
  if (!K_host || !V_host) return fail(h, HERMES_EINVAL, "K_new / V_new must not be NULL");
  const hermes_config& c = h->cfg;
  if (n_new <= 0 || n_new > c.max_chunk_tokens) return fail(h, HERMES_EINVAL, "n_new = %d not in [1, %d] (host path)", n_new, c.max_chunk_tokens);
  if (h->lb && kept_out_host) return fail(h, HERMES_EINVAL, "kept_out is not available with layer-dependent budgets (use hermes_get_cache)");
  if (Q_host && (n_probe <= 0 || n_probe > c.max_probe_tokens)) return fail(h, HERMES_EINVAL, "n_probe = %d not in [1, %d]", n_probe, c.max_probe_tokens);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const size_t BL = size_t(c.n_streams) * c.n_layers;
  const size_t kv_bytes = BL * n_new * h->lay.row_bytes;
  // Two staging sets: the copies of this call run on the library's copy stream while the kernels of the previous call (on
  // the caller's stream) still read the other set.  Q and K go first, V last: the scoring kernels, which never read V,
  // start as soon as K is across, and the V rows are appended behind an event wait.
  const int p = int(h->host_calls & 1u);
  char* sk = h->ws + h->lay.stage_k + p * h->lay.stage_kv_bytes;
  char* sv = h->ws + h->lay.stage_v + p * h->lay.stage_kv_bytes;
  char* sq = h->ws + h->lay.stage_q + p * h->lay.stage_q_bytes;
  if (!h->side_stream) {
    CUDA_TRY(h, cudaStreamCreateWithFlags(&h->side_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_k_done[i], cudaEventDisableTiming));
      CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_v_done[i], cudaEventDisableTiming));
      CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_free[i], cudaEventDisableTiming));
    }
  }
  cudaStream_t cs = h->side_stream;
  if (h->ev_free_set[p]) CUDA_TRY(h, cudaStreamWaitEvent(cs, h->ev_free[p], 0));   // the call before the last is done with set p
  if (Q_host) {
    // the probe slices of shallow layers are never read (include/hermes.h): per stream, copy layers [n_shallow, L) only
    const size_t lq = size_t(c.n_q_heads) * n_probe * c.head_dim * h->lay.esize, ns = size_t(h->lay.n_shallow);
    if (c.n_layers > int(ns))
      CUDA_TRY(h, cudaMemcpy2DAsync(sq + ns * lq, c.n_layers * lq, static_cast<const char*>(Q_host) + ns * lq, c.n_layers * lq,
                                    (c.n_layers - ns) * lq, size_t(c.n_streams), cudaMemcpyHostToDevice, cs));
  }
  CUDA_TRY(h, cudaMemcpyAsync(sk, K_host, kv_bytes, cudaMemcpyHostToDevice, cs));
  CUDA_TRY(h, cudaEventRecord(h->ev_k_done[p], cs));
  CUDA_TRY(h, cudaMemcpyAsync(sv, V_host, kv_bytes, cudaMemcpyHostToDevice, cs));
  CUDA_TRY(h, cudaEventRecord(h->ev_v_done[p], cs));
  CUDA_TRY(h, cudaStreamWaitEvent(s, h->ev_k_done[p], 0));
  ++h->host_calls;
  const int len_before = h->len;
  int rc = append_impl(h, sk, sv, Q_host ? sq : nullptr, n_new, n_probe, pos_start, cuda_stream, h->ev_v_done[p]);
  if (rc != HERMES_OK) {                               // nothing was enqueued: still join the copy stream
    cudaStreamWaitEvent(s, h->ev_v_done[p], 0);
    return rc;
  }
  CUDA_TRY(h, cudaEventRecord(h->ev_free[p], s));
  h->ev_free_set[p] = true;
  const bool evicted = Q_host && len_before + n_new > c.budget;
  if (kept_out_host && evicted)
    CUDA_TRY(h, cudaMemcpyAsync(kept_out_host, h->geom.kept, BL * c.budget * 4, cudaMemcpyDeviceToHost, s));
  return HERMES_OK;
}
