// hermes_topk_noalloc -- Eq. 6 Top-K of ONE score vector, for callers that may not allocate:
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The entry point takes
// no handle and no workspace: the scratch of the selection (orderable keys, digit histograms, chunk prefixes)
// lives in a file-scope device array of kTopkScratchBytes (268 KB) that every GPU loading this library holds
// until the process exits.
//
// A variant of k_select's a4 stage (k_select.cuh): same total order (score, index), ties evict the smaller
// index, kept indices emitted ascending -- so its output is bit-identical to the handle path's kept list for
// the same scores.  The handle path keeps the scores in dynamic shared memory and its prefixes in the caller's
// workspace; here they sit in the static array.  Self-contained on purpose: this translation unit shares no
// kernel with hermes_api.cu, and no existing code path changes.
//
// The array is shared by every call of the process on that GPU and keeps the last call's contents: the kernel
// clears the digit histograms (the only part that must start at zero) itself, everything else is written
// before it is read.  Two calls that OVERLAP on the GPU (different streams, no ordering between them) race on
// it; calls on one stream, or ordered by events, are safe.
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include <cstdio>
#include <mutex>

#include "../../include/hermes.h"

namespace hk_noalloc {

constexpr int kTopkMaxTokens = 65536;                 // largest score vector
constexpr int kTopkThreads = 1024;
constexpr int kTopkChunks = kTopkMaxTokens / 32;      // 32-token chunks of the flag scan
constexpr int kOffKeys = 0;                           // [kTopkMaxTokens] orderable keys
constexpr int kOffChunk = kOffKeys + kTopkMaxTokens;  // [kTopkChunks] packed (#less | #equal << 16) exclusive prefixes
constexpr int kOffHist = kOffChunk + kTopkChunks;     // [4 rounds][256] digit histograms -- must start at zero
constexpr int kScratchWords = kOffHist + 4 * 256;
constexpr size_t kTopkScratchBytes = size_t(kScratchWords) * 4;
static_assert(kTopkScratchBytes == 274432, "the size include/hermes.h and README.md state");

// In host code this name is a host-side stand-in, NOT a device address: only cudaGetSymbolAddress() (below)
// yields the pointer a kernel can take.
static __device__ __align__(256) uint32_t g_topk_scratch[kScratchWords];

__device__ __forceinline__ uint32_t orderable_key(float f) {     // monotone float -> uint32 map
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// One thread block.  scratch = device address of g_topk_scratch.
__global__ void __launch_bounds__(kTopkThreads)
k_topk_static(const float* __restrict__ scores, int T, int k, int32_t* __restrict__ kept, uint32_t* scratch) {
  __shared__ int whist[32 * 256];                     // warp-private digit histograms
  __shared__ uint32_t warp_tot[33];
  __shared__ uint32_t sel_prefix;
  __shared__ int sel_remaining;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t* keys = scratch + kOffKeys;
  uint32_t* chunk_pre = scratch + kOffChunk;
  uint32_t* hist = scratch + kOffHist;

  // the array keeps the last call's contents: the histograms are accumulated with atomics and must start at zero
  __stcg(hist + tid, 0u);                             // 4 x 256 = 1024 counters, one per thread
  for (int i = tid; i < 32 * 256; i += kTopkThreads) whist[i] = 0;
  for (int i = tid; i < T; i += kTopkThreads) __stcg(keys + i, orderable_key(__ldg(scores + i)));
  if (tid == 0) { sel_prefix = 0u; sel_remaining = T - k; }      // evict the T - k smallest
  __syncthreads();                                    // block-wide: the global stores above are visible to the block

  // ---- radix select of the (T-k)-th smallest key, 8 bits per round, MSB first -----------------------
  for (int round = 0; round < 4; ++round) {
    const int shift = 24 - 8 * round;
    const uint32_t himask = round == 0 ? 0u : (0xFFFFFFFFu << (shift + 8));
    const uint32_t prefix = sel_prefix;
    int* my_hist = whist + warp * 256;
    for (int i = tid; i < T; i += kTopkThreads) {
      const uint32_t key = __ldcg(keys + i);
      if ((key & himask) == prefix) atomicAdd(&my_hist[(key >> shift) & 255u], 1);
    }
    __syncthreads();
    {                                                 // fold 8 warp histograms per thread into the round's global histogram
      const int q = tid >> 8, d = tid & 255;
      int c = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) { c += whist[(q * 8 + w) * 256 + d]; whist[(q * 8 + w) * 256 + d] = 0; }
      if (c) atomicAdd(hist + round * 256 + d, uint32_t(c));
    }
    __syncthreads();
    if (warp == 0) {                                  // the bucket that holds the (T-k)-th smallest
      int c[8], tot = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) { c[j] = int(__ldcg(hist + round * 256 + lane * 8 + j)); tot += c[j]; }
      int inc = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
      }
      const int rem = sel_remaining;
      __syncwarp();
      int below = inc - tot;
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
  const uint32_t vstar = sel_prefix;                  // key of the (T-k)-th smallest score (0 when k == T)
  const int r_eq = sel_remaining;                     // evicted among keys == vstar: the smallest indices

  // ---- flags + exclusive scan over 32-token chunks; kept indices leave in ascending order -----------
  const int n_chunks = (T + 31) >> 5;
  for (int c = warp; c < n_chunks; c += 32) {
    const int i = c * 32 + lane;
    const uint32_t key = i < T ? __ldcg(keys + i) : 0xFFFFFFFFu;
    const uint32_t lt = __ballot_sync(0xffffffffu, i < T && key < vstar);
    const uint32_t eq = __ballot_sync(0xffffffffu, i < T && key == vstar);
    if (lane == 0) __stcg(chunk_pre + c, uint32_t(__popc(lt)) | (uint32_t(__popc(eq)) << 16));
  }
  __syncthreads();
  {
    // both 16-bit halves of every EXCLUSIVE prefix stay below 65536 (at most T - 32 tokens precede a chunk)
    const int cpt = (n_chunks + kTopkThreads - 1) / kTopkThreads;          // <= 2
    const int c_beg = min(tid * cpt, n_chunks), c_end = min(c_beg + cpt, n_chunks);
    uint32_t mine = 0;
    for (int c = c_beg; c < c_end; ++c) mine += __ldcg(chunk_pre + c);
    uint32_t inc = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t n = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += n;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      const uint32_t w = warp_tot[lane];
      uint32_t winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t n = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) winc += n;
      }
      warp_tot[lane] = winc - w;
    }
    __syncthreads();
    uint32_t run = warp_tot[warp] + inc - mine;
    for (int c = c_beg; c < c_end; ++c) { const uint32_t v = __ldcg(chunk_pre + c); __stcg(chunk_pre + c, run); run += v; }
  }
  __syncthreads();
  const uint32_t lane_lt = (1u << lane) - 1u;
  for (int c = warp; c < n_chunks; c += 32) {
    const int i = c * 32 + lane;
    const uint32_t key = i < T ? __ldcg(keys + i) : 0xFFFFFFFFu;
    const uint32_t lt = __ballot_sync(0xffffffffu, i < T && key < vstar);
    const uint32_t eq = __ballot_sync(0xffffffffu, i < T && key == vstar);
    const uint32_t pre = __ldcg(chunk_pre + c);
    const int lt_before = int(pre & 0xFFFFu) + __popc(lt & lane_lt);
    const int eq_before = int(pre >> 16) + __popc(eq & lane_lt);
    const bool evict = key < vstar || (key == vstar && eq_before < r_eq);
    if (i < T && !evict) kept[i - lt_before - min(eq_before, r_eq)] = i;
  }
}

// ---- host side -----------------------------------------------------------------------------------------
constexpr int kMaxDevices = 64;
static std::atomic<uint32_t*> g_scratch_ptr[kMaxDevices];   // device address of g_topk_scratch, per device ordinal
static std::mutex g_setup_mu;
static thread_local char t_err[256] = "";

static int fail(int code, const char* fmt, long long a = 0, long long b = 0) {
  std::snprintf(t_err, sizeof t_err, fmt, a, b);
  return code;
}

// Resolves the scratch address on the CURRENT device (once per device); no allocation: the array is part of the
// loaded module.
static int scratch_of_current_device(uint32_t** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { std::snprintf(t_err, sizeof t_err, "cudaGetDevice: %s", cudaGetErrorString(e)); return HERMES_ECUDA; }
  if (dev < 0 || dev >= kMaxDevices) return fail(HERMES_EINVAL, "device ordinal %lld outside [0, %lld)", dev, kMaxDevices);
  uint32_t* p = g_scratch_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    std::lock_guard<std::mutex> lock(g_setup_mu);
    p = g_scratch_ptr[dev].load(std::memory_order_relaxed);
    if (!p) {
      void* sym = nullptr;
      e = cudaGetSymbolAddress(&sym, g_topk_scratch);        // with `dev` current: the address is per device
      if (e != cudaSuccess || !sym) {
        (void)cudaGetLastError();
        std::snprintf(t_err, sizeof t_err, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
        return HERMES_ECUDA;
      }
      p = static_cast<uint32_t*>(sym);
      g_scratch_ptr[dev].store(p, std::memory_order_release);
    }
  }
  *out = p;
  return HERMES_OK;
}

}  // namespace hk_noalloc

extern "C" {

int32_t hermes_topk_noalloc_max_tokens(void) { return hk_noalloc::kTopkMaxTokens; }

const char* hermes_topk_noalloc_error(void) { return hk_noalloc::t_err; }

int hermes_topk_noalloc_setup(void) {
  uint32_t* p = nullptr;
  return hk_noalloc::scratch_of_current_device(&p);
}

int hermes_topk_noalloc(const float* scores, int32_t n_tokens, int32_t k, int32_t* kept_out, void* cuda_stream) {
  using namespace hk_noalloc;
  if (!scores || !kept_out) return fail(HERMES_EINVAL, "scores and kept_out must be device pointers, not NULL");
  if (n_tokens < 1) return fail(HERMES_EINVAL, "n_tokens = %lld must be >= 1", n_tokens);
  if (n_tokens > kTopkMaxTokens)
    return fail(HERMES_ECAPACITY, "n_tokens = %lld exceeds the static scratch maximum of %lld tokens", n_tokens, kTopkMaxTokens);
  if (k < 1 || k > n_tokens) return fail(HERMES_EINVAL, "k = %lld must lie in [1, n_tokens = %lld]", k, n_tokens);
  uint32_t* scratch = nullptr;
  const int rc = scratch_of_current_device(&scratch);
  if (rc != HERMES_OK) return rc;
  k_topk_static<<<1, kTopkThreads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(scores, n_tokens, k, kept_out, scratch);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    std::snprintf(t_err, sizeof t_err, "k_topk_static launch: %s", cudaGetErrorString(e));
    return HERMES_ECUDA;
  }
  return HERMES_OK;
}

}  // extern "C"
