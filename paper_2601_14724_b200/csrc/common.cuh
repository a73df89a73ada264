// Shared device-side definitions for the HERMES update kernels (sm_100a).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace hk {

constexpr float kLog2e = 1.4426950408889634f;
constexpr int kMaxLayers = 256;

// Geometry + workspace pointers, passed by value to every kernel.
struct Geom {
  int B, L, Hq, Hkv, G, d;
  int cap;          // slots per layer slab
  int budget;       // |M|
  int n_axes;       // 1 (1D RoPE) or 3 (M-RoPE)
  int row_elems;    // Hkv * d elements per token row
  int n_shallow;    // layers [0, n_shallow) are pure recency (Eq. 1) and are not scored
  int n_deep;       // layers [L - n_deep, L) are the deep stage
  int probe_deep_begin; // deep layers use probe rows [begin, P) only (hybrid guidance, DESIGN f3)
  int summary;      // 1: deep layers keep budget-1 tokens and append one summary token (Alg. 1)
  int n_evict_max;  // capacity of the evicted index lists: cap - budget + 1
  int p_max;        // max probe tokens (row capacity of the stat buffers = Hq * p_max)
  int pos_offset;
  int sec_t, sec_h; // M-RoPE: pairs [0,sec_t) -> t, [sec_t, sec_t+sec_h) -> h, rest -> w
  int compact_axes;
  int grid_h, grid_w;
  int table_rows;   // rotary table covers delta in [-(table_rows-1), 0]
  int n_vh_max;     // column-sum slots per (stream, layer): Hkv * max row super-chunks per KV head
  void* kc;         // K cache   [B*L*2][cap][row_elems]
  void* vc;         // V cache   same
  int32_t* posc;    // positions [B*L*2][n_axes][cap]
  float* colsum;    // [B*L][n_vh_max][cap] per-(KV head, row super-chunk) column sums of the softmax (a1)
  float* wsum;      // [B*L][cap] W_i: column sums added over KV heads / (Hq*P)  (Eq. 2)
  uint32_t* wmax;   // [B*L] max_i W_i as float bits (W >= 0), zeroed by k_append
  float* rowstat;   // [B*L][Hq*p_max][2] (m2, 1/Z) per probe row, log2 domain
  float* partial;   // partial (m2, z) of pass 1: SIMT path [B*L][Hq*p_max][n_part][2]; tcgen05 path [B*L][n_slot][Hq*p_max][2]
  float* scores;    // [B*L][cap]  smoothed scores S~ of the last eviction (a3)
  int32_t* kept;    // [B*L][budget] ascending kept indices I_l (a4)
  int32_t* delta;   // [B*L][n_axes][budget] p_new - p_old of every kept token (a6 -> a7)
  int32_t* evicted; // [B*L][n_evict_max] ascending evicted indices (summary-token layers only)
  float2* rope_tab; // [table_rows][d/2] (cos, sin)(-r * theta_j) for r = row index
  double* rope_freq;// [d/2] theta_j in fp64 (slow path for deltas outside the table)
  float2* sum_tab;  // summary tokens: [sum_tab_rows][d/2] (cos, sin)(delta * theta_j), delta = row - sum_tab_zero
  int sum_tab_zero; // row of delta = 0 in sum_tab
  int sum_tab_rows;
  float* omega;     // [L] weight of the recency term (Eq. 3-4); 1 shallow, 0 deep
  float* lambda;    // [L] Eq. 7
  int32_t* status;  // sticky device status word
  unsigned* seg_cnt;// [B*L*n_vh_max] tcgen05 scoring: pass-1 progress per group, zeroed by k_append
  // layer-dependent budgets (DESIGN f4); both NULL otherwise.  Rewritten by a stream-ordered copy before every update.
  const int32_t* lay_T;    // [L] candidates T_l = len_l + n_new of this update
  const int32_t* lay_keep; // [L] tokens layer l holds after this update: m_l if T_l > m_l (it compresses), else T_l
};

// Candidates / retained tokens of layer l in this update (uniform: the kernel's scalar arguments).
__device__ __forceinline__ int layer_T(const Geom& g, int l, int Tn) { return g.lay_T ? __ldg(g.lay_T + l) : Tn; }
__device__ __forceinline__ int layer_keep(const Geom& g, int l) { return g.lay_keep ? __ldg(g.lay_keep + l) : g.budget; }

__host__ __device__ inline size_t slab_index(const Geom& g, int b, int l, int buf) {
  return (size_t(b) * g.L + l) * 2 + buf;
}

// ---- element traits --------------------------------------------------------------------------
template <typename T> struct Elem;
template <> struct Elem<float> {
  static constexpr int kPerVec = 4;  // elements per 16-byte vector
  __device__ static inline void unpack(const uint4& v, float* f) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y);
    f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
  __device__ static inline uint4 pack(const float* f) {
    return make_uint4(__float_as_uint(f[0]), __float_as_uint(f[1]), __float_as_uint(f[2]), __float_as_uint(f[3]));
  }
  __device__ static inline float to_float(float x) { return x; }
};
template <> struct Elem<__nv_bfloat16> {
  static constexpr int kPerVec = 8;
  __device__ static inline void unpack(const uint4& v, float* f) {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      f[2 * i] = __uint_as_float(w[i] << 16);
      f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
  }
  __device__ static inline uint4 pack(const float* f) {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      // round-to-nearest-even fp32 -> bf16 (cvt.rn.bf16x2.f32 packs hi:lo)
      __nv_bfloat162 p = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);
      w[i] = *reinterpret_cast<uint32_t*>(&p);
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
  }
  __device__ static inline float to_float(__nv_bfloat16 x) { return __bfloat162float(x); }
};

__device__ inline uint4 ldg_stream(const void* p) {  // streaming 128-bit load, no L1 allocation
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ inline void stg_stream(void* p, const uint4& v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
               :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// 2^x on the MUFU pipe (ex2.approx.ftz: rel. error <= 2^-22, ex2(-inf) = +0); exp2f() costs 4 instructions
__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// Programmatic dependent launch: every kernel of an update is launched with the programmatic-stream-
// serialization attribute, so its CTAs may become resident (and run their prologue) while the previous
// kernel drains.  pdl_wait() blocks until the previous kernel has completed and its writes are visible;
// data written by earlier kernels is then read with ld.global.cg (L2), never through a possibly stale L1 line.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ inline float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ inline float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

}  // namespace hk
