/*
 * hermes.h -- C ABI of the B200-native HERMES per-chunk hierarchical KV-cache update
 *             (arXiv 2601.14724; citations are PAPER.md:<line> + equation).
 *
 * One call of hermes_append_chunk() is one chunk arrival (Fig. 3 at :61):
 *   a0 append the chunk's K/V after the cached tokens of every layer;
 *   a1 attention importance W of every cached video token w.r.t. the guidance-prompt
 *      pseudo-query (Eq. 2), middle + deep layers only;
 *   a2 normalise, recency (Eq. 1) and layer weighting (Eq. 3-4);
 *   a3 cross-layer memory smoothing (Eq. 5; lambda of Eq. 7);
 *   a4 per-layer Top-K under the budget |M| (Eq. 6);
 *   a5 gather-compaction K_l[I_l], V_l[I_l] (Eq. 6);
 *   a6 eager position re-indexing (Eq. 8; M-RoPE Eq. 11);
 *   a7 delta rotary correction of the kept keys (Eq. 9-10; Eq. 12-13, :629-634).
 * Every step runs in sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *   - All functions return HERMES_OK (0) or a negative hermes_status; they never throw, abort or print.
 *   - "device pointer" = memory of the CUDA device in hermes_config.device; "host pointer" = CPU memory.
 *   - Tensors are dense, row-major, element type hermes_config.dtype (fp32 or bf16).
 *   - Calls are stream-ordered and asynchronous: they enqueue work on `cuda_stream` (a cudaStream_t;
 *     NULL = the legacy default stream) and return; no host synchronisation on the success path.
 *     Caller buffers must stay valid and unmodified until the stream has passed the call.
 *   - The library allocates no device memory: the caller provides one workspace of
 *     hermes_workspace_bytes() bytes (256-byte aligned), which the handle owns until hermes_destroy().
 *   - Query head h uses KV head h / (n_q_heads / n_kv_heads) (grouped-query attention).
 *   - A handle is not thread-safe; use one per host thread or serialise calls.
 *   - hermes_append_chunk() with uniform budgets enqueues kernels only (no copy, no allocation, no host synchronisation), so it
 *     may be called on a capturing stream.  The handle's host-side state advances when the call is made, not when the graph
 *     runs: capture in steady state (eager re-indexing, len == budget, default pos_start, fixed n_new / n_probe) and an EVEN
 *     number of updates (the double buffer flips once per evicting update); such a graph can be replayed with new data
 *     in the same input buffers, and hermes_get_cache() stays valid after any number of replays.
 *   - The tcgen05 scoring kernel is persistent (at most one CTA per SM) and a CTA's second pass waits for row
 *     statistics written by other CTAs of the same launch, so every CTA of its grid must be resident at once.  It is
 *     launched cooperatively: on a device partition that cannot hold the grid (MPS active-thread percentage, a green
 *     context) the runtime refuses the launch, and the handle scores on the CUDA-core path from then on
 *     (HERMES_ECUDA if score_path forces tcgen05).
 */
#ifndef HERMES_H_
#define HERMES_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  HERMES_OK = 0,
  HERMES_EINVAL = -1,     /* bad argument / unsupported geometry; state unchanged            */
  HERMES_ECAPACITY = -2,  /* len + n_new exceeds max_tokens (or workspace too small)          */
  HERMES_ESTATE = -3,     /* call not valid in the handle's current state                     */
  HERMES_ECUDA = -4,      /* a CUDA runtime / driver call failed (no device, launch error...) */
  HERMES_ENOMEM = -5      /* host allocation failed                                           */
} hermes_status;

enum { HERMES_F32 = 0, HERMES_BF16 = 1 };
enum { HERMES_ROPE_1D = 0, HERMES_ROPE_M3D = 1 };   /* App. E.1 / App. E.2                    */
enum { HERMES_NORM_MAX = 0, HERMES_NORM_SUM = 1 };  /* alpha of Eq. 1/2 (DESIGN c2)           */
enum { HERMES_SCORE_AUTO = 0, HERMES_SCORE_SIMT = 1, HERMES_SCORE_TCGEN05 = 2 };
enum { HERMES_REINDEX_EAGER = 0, HERMES_REINDEX_LAZY = 1 };   /* Sec. 3.3   */

typedef struct hermes hermes_t;  /* opaque; owns n_streams x n_layers double-buffered caches   */

typedef struct {
  int32_t n_layers, n_q_heads, n_kv_heads;
  int32_t head_dim;             /* 32, 64 or 128                                              */
  int32_t dtype;                /* HERMES_F32 | HERMES_BF16: K, V and Q_probe element type     */
  int32_t n_streams;            /* B independent streams advanced by every call                */
  int32_t tokens_per_frame;     /* N_f; informational                                          */
  int32_t budget;               /* |M| tokens kept per layer                    */
  int32_t max_chunk_tokens;     /* largest n_new (binding for the host entry point and for LAZY re-indexing; an
                                   append through hermes_append_chunk is otherwise bounded by max_tokens only) */
  int32_t max_tokens;           /* slots per layer; 0 -> budget + max_chunk_tokens             */
  int32_t max_probe_tokens;     /* largest n_probe                                             */
  int32_t n_shallow, n_deep;    /* -1 -> max(1, round(0.1 L)), max(1, round(0.3 L)) */
  int32_t l_short, l_long;      /* -1 -> first / last middle layer (Eq. 3)                     */
  float omega0, gamma;          /* Eq. 3: 0.75, 0.6                              */
  float forget_rate;            /* k > 0 of Eq. 1, per token of temporal distance              */
  int32_t norm_mode;            /* HERMES_NORM_*                                               */
  float lambda_shallow, lambda_middle, lambda_deep; /* Eq. 7: 0.1, 0.3, 0.4                    */
  float softmax_scale;          /* 0 -> 1/sqrt(head_dim)                                       */
  int32_t rope_mode;            /* HERMES_ROPE_*                                               */
  float rope_theta;             /* RoPE base; theta_j = base^(-2j/head_dim)                    */
  int32_t mrope_section[3];     /* rotary pairs owned by (t, h, w); sum = head_dim/2           */
  int32_t mrope_compact_axes;   /* bit0 t, bit1 h, bit2 w: axes re-indexed by Eq. 11           */
  int32_t mrope_grid_h, mrope_grid_w; /* merged patch grid; tokens per temporal step = h*w     */
  int32_t pos_offset;           /* length of the fixed system prefix            */
  int32_t reindex_mode;         /* HERMES_REINDEX_*: EAGER re-indexes at every compression step;
                                   LAZY keeps original indices (kept keys are copied, not rotated) and
                                   re-indexes only at the step after which the next chunk (max_chunk_tokens
                                   positions; M-RoPE: its temporal steps) would exceed max_position        */
  int32_t max_position;         /* LAZY: the model's position limit (> pos_offset + budget + chunk span) */
  int32_t probe_deep_begin;     /* deep layers score with probe rows [begin, n_probe) only: Q_probe rows are
                                   [local prompt | global prompt], middle layers use all (App. B);
                                   0 = all rows everywhere                                              */
  int32_t summary_token;        /* 1: every deep layer keeps budget-1 tokens by Top-K and appends ONE summary
                                   token of the evicted ones (Alg. 1) in slot budget-1;
                                   last_kept[budget-1] = -1 marks it.  Its position: pos_offset+budget-1 at a step that
                                   re-indexes; under LAZY re-indexing, between re-index steps, the position after the
                                   newest token (the next chunk then starts one position later).  Needs HERMES_ROPE_1D  */
  float budget_weight[3];       /* layer-dependent budgets (Tab. 5): weight of a shallow / middle / deep
                                   layer.  With the total budget * n_layers fixed, layer i keeps
                                   m_i = floor(w_i / sum_j w_j * budget * n_layers) tokens, the residue goes to the last
                                   layer.  {1, 1, 1} (default): `budget` everywhere.  Unequal weights need HERMES_ROPE_1D;
                                   with summary_token a deep layer i keeps m_i - 1 tokens + its summary token     */
  int32_t defer_v;              /* 1 (default): on the tcgen05 path an eviction compacts K at once but leaves the
                                   kept V rows to be moved by the NEXT update's scoring kernel (V is not read by
                                   scoring, so the copy hides behind it); hermes_get_cache() and updates that do
                                   not score on tcgen05 first run the pending move on their own.  0: never defer */
  int32_t score_path;           /* HERMES_SCORE_*: AUTO picks tcgen05 when the contraction is dense */
  int32_t device;               /* CUDA device ordinal                                         */
} hermes_config;

/* Borrowed DEVICE pointers into the workspace for one (stream, layer); valid until the next
 * hermes_append_chunk*() or hermes_destroy() on the handle.  Contents are defined once the stream of the
 * last append has been synchronised.                                                                  */
typedef struct {
  const void *k, *v;            /* [len, n_kv_heads, head_dim], token-major                    */
  const int32_t *pos;           /* [n_axes][pos_stride]; first `len` entries of each axis valid */
  int32_t n_axes;               /* 1 (1D RoPE) or 3 (M-RoPE: t, h, w)                          */
  int32_t pos_stride;
  int32_t len;                  /* host-tracked: min(tokens appended, this layer's budget) after an eviction */
  const float *last_scores;     /* [last_T] smoothed scores S~ of the last eviction, else NULL  */
  const int32_t *last_kept;     /* [len] ascending indices I_l into the last candidate list      */
  int32_t last_T;               /* this layer's candidates at the last eviction (0 if none yet)  */
} hermes_cache_view;

/* Defaults of the paper for everything but geometry; geometry fields are 0. */
void hermes_default_config(hermes_config *cfg);

/* Bytes of device workspace a handle with this config needs; 0 if the config is invalid.              */
size_t hermes_workspace_bytes(const hermes_config *cfg);

/* Per-layer budgets m_i of a config (hermes_config.budget_weight): writes min(n, n_layers) values to out
 * and returns n_layers, or HERMES_EINVAL for an invalid config.  Host-only: needs no device.                         */
int hermes_layer_budgets(const hermes_config *cfg, int32_t *out, int32_t n);

/* Validates cfg (HERMES_EINVAL: H_q % H_kv != 0, head_dim not in {32,64,128}, sum(mrope_section) !=
 * head_dim/2, budget <= 0, forget_rate <= 0, n_shallow + n_deep > L, ...), binds `workspace`
 * (device pointer, `bytes` >= hermes_workspace_bytes, else HERMES_ECAPACITY), builds the rotary table
 * on `cfg->device`.  HERMES_ECUDA if no usable sm_100 device.  *out is NULL on failure.
 * This call synchronises the device once.                                                            */
int hermes_create(const hermes_config *cfg, void *workspace, size_t bytes, hermes_t **out);

/* One chunk arrival for all B streams.
 *   K_new, V_new : device, [B, L, n_new, H_kv, d]; K is post-RoPE at the arrival positions.
 *   Q_probe      : device, [B, L, H_q, n_probe, d] post-RoPE guidance-prompt query states, or NULL.
 *                  Slices of shallow layers are never read.
 *   pos_start    : 1D: position of the chunk's token 0 (token j sits at pos_start + j); M-RoPE: temporal
 *                  index of the chunk's first step.  -1 -> default: 1D pos_offset + len; M-RoPE
 *                  pos_offset + min(temporal steps seen, budget).  Must exceed every cached position.
 * With T = len + n_new: if Q_probe == NULL or T <= budget the chunk is only appended;
 * otherwise steps a1-a7 run and len becomes budget.  T > max_tokens -> HERMES_ECAPACITY, state unchanged. */
int hermes_append_chunk(hermes_t *h, const void *K_new, const void *V_new, const void *Q_probe,
                        int32_t n_new, int32_t n_probe, int32_t pos_start, void *cuda_stream);

/* Same update with HOST buffers (pinned memory recommended), which must hold their data when the call is made: Q_probe
 * (the slices of the scored layers only), K_new and then V_new are copied to the device with cudaMemcpyAsync on a
 * library-owned copy stream (created on first use) into one of two staging sets, so the copies of a call overlap the kernels of the call before it; `cuda_stream`
 * waits for K before the update's kernels and for V before the V rows are appended, so everything the call enqueues is
 * ordered on `cuda_stream` when it returns.  If kept_out != NULL, copies the kept index lists I_l [B, L, budget] int32
 * back to the host on `cuda_stream` (only meaningful when an eviction ran; not available with layer-dependent budgets).
 * The host buffers must stay valid until `cuda_stream` has passed the call.                                           */
int hermes_append_chunk_host(hermes_t *h, const void *K_new_host, const void *V_new_host,
                             const void *Q_probe_host, int32_t n_new, int32_t n_probe,
                             int32_t pos_start, int32_t *kept_out_host, void *cuda_stream);

/* Fills *out for (stream, layer).  No synchronisation; if a V compaction is pending (defer_v) it is enqueued
 * on the stream of the last append first.                                                              */
int hermes_get_cache(hermes_t *h, int32_t stream, int32_t layer, hermes_cache_view *out);

/* Host-tracked token count per layer (same for every stream; with layer-dependent budgets the largest layer's). */
int32_t hermes_len(const hermes_t *h);

/* Host-tracked token count of one layer (differs from hermes_len only with layer-dependent budgets); -1 if out of range. */
int32_t hermes_layer_len(const hermes_t *h, int32_t layer);

/* Budget m_i of one layer (hermes_config.budget unless budget_weight is unequal); -1 if out of range.            */
int32_t hermes_layer_budget(const hermes_t *h, int32_t layer);

/* Device-side sticky status word, read with a blocking copy: 0 = ok; bit0 = M-RoPE coordinate range
 * too wide to compact, bit1 = rotary delta outside the table (slow path taken; results still valid).  */
int hermes_device_status(hermes_t *h, int32_t *status_out);

/* Per-kernel timing: when enabled, CUDA events bracket each kernel of the next append calls.
 * hermes_get_profile() synchronises on the last call's events and writes up to n kernel durations in
 * milliseconds, in HERMES_K_* order (0 for kernels that did not run); returns the count written.      */
enum { HERMES_K_APPEND = 0, HERMES_K_SCORE_STATS = 1, HERMES_K_SCORE_COMBINE = 2,
       HERMES_K_SCORE_COLSUM = 3, HERMES_K_SELECT = 4, HERMES_K_GATHER = 5, HERMES_K_SUMMARY = 6, HERMES_K_COUNT = 7 };
int hermes_set_profiling(hermes_t *h, int32_t enable);
int hermes_get_profile(hermes_t *h, float *ms_out, int32_t n);

/* Which scoring path the last eviction used: HERMES_SCORE_SIMT or HERMES_SCORE_TCGEN05 (0 if none).  */
int32_t hermes_last_score_path(const hermes_t *h);

/* 1 if a V compaction is pending (defer_v): the kept V rows of the last eviction have not been moved yet.        */
int32_t hermes_v_pending(const hermes_t *h);

/* Number of kernels launched by the last append call.                                                */
int32_t hermes_last_launch_count(const hermes_t *h);

void hermes_destroy(hermes_t *h);

/* Message of the last failing call on this handle (or of the last failing hermes_create if h == NULL). */
const char *hermes_last_error(const hermes_t *h);

/* ---- allocation-free Top-K (csrc/hermes_noalloc.cu) --------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): Eq. 6 on ONE score vector, with no handle and no workspace.  Its scratch (268 KB: sortable
 * keys, digit histograms, scan prefixes) is a file-scope static device array that every GPU loading the library holds
 * until the process exits, hence the size limit below.
 *   scores   : device, [n_tokens] fp32 (e.g. hermes_cache_view.last_scores); not modified.
 *   kept_out : device, [k] int32; receives the indices of the k largest scores in ASCENDING index order.  Total order
 *              (score, index): among equal scores the smaller index is evicted first -- the rule of the update path,
 *              so for the same scores the result equals hermes_cache_view.last_kept bit for bit.
 * Runs on the CURRENT device (cudaSetDevice); `cuda_stream` must belong to it.  Asynchronous: one kernel is enqueued.
 * Errors: HERMES_EINVAL (NULL pointer, n_tokens < 1, k outside [1, n_tokens]); HERMES_ECAPACITY (n_tokens above the
 * maximum of 65 536 reported by the max_tokens query below); HERMES_ECUDA (CUDA call failed).  The message is
 * thread-local and read with the error query below.
 * The call allocates nothing on host or device.  The first call on a device resolves the array's device address
 * (cudaGetSymbolAddress, once per device); callers that capture graphs make that happen before capture with the
 * setup call, on the device they will use.
 * Every call on a GPU shares the one array: calls ordered on a stream (or by events) are safe, calls that OVERLAP on
 * the GPU race on it and return garbage.                                                                           */
int hermes_topk_noalloc(const float *scores, int32_t n_tokens, int32_t k, int32_t *kept_out, void *cuda_stream);
int hermes_topk_noalloc_setup(void);           /* resolve the scratch address on the current device; HERMES_OK / _ECUDA */
int32_t hermes_topk_noalloc_max_tokens(void);  /* 65536 */
const char *hermes_topk_noalloc_error(void);   /* message of this thread's last failing no-alloc call ("" if none)    */

#ifdef __cplusplus
}
#endif
#endif /* HERMES_H_ */
