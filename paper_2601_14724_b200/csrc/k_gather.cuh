// a5 + a7 fused -- gather-compaction K_l[I_l], V_l[I_l] (Eq. 6) with the delta rotary
// correction of the kept keys (Eq. 9-10; M-RoPE Eq. 12-13), from the
// current buffer into the other one.  HBM-bound: every thread moves 4 x 16 bytes per step (K lo/hi halves
// of a rotary pair group + the same two vectors of V), 128-bit coalesced, streaming cache policy; the
// kept index and the position deltas of the NEXT step are prefetched while the current one is in flight.
// Measured and not adopted (configs[1], K-only launch 68 us, pure copy under lazy re-indexing 57 us): table row requested
// before the keys are unpacked (spills at 64 registers: 78 us); keys staged one trip ahead through thread-private shared
// memory by cp.async (85 us; pure copy 68); rows moved by 1D bulk copies through a shared-memory ring and rotated in place
// (79 us with the table read by __ldg, 111 us with the table row bulk-copied beside the key row; pure copy 56 us);
// prefetch.global.L1 of the next trip's table slice (CCTL.PF1: 2 x slower).
//
// A "unit" = kPerVec rotary pairs of one KV head: elements [j0, j0+kPerVec) and [j0+d/2, ...) of the head.
// Rotation: angle table (cos, sin)(delta * theta_j) built in fp64 at create time; fp32 products and
// sums WITHOUT fused multiply-add, round-to-nearest-even to the storage dtype; delta = 0 is a bit-exact
// copy (DESIGN c14).  Deltas outside the table take an fp64 sincos slow path (status bit 1).
#pragma once
#include "common.cuh"

namespace hk {

constexpr int kGatherThreads = 256;

__device__ __forceinline__ void rot_pair(float& x, float& y, float c, float s) {
  const float xn = __fsub_rn(__fmul_rn(x, c), __fmul_rn(y, s));
  const float yn = __fadd_rn(__fmul_rn(x, s), __fmul_rn(y, c));
  x = xn; y = yn;
}

__device__ __noinline__ float2 slow_cos_sin(const double* freq, int32_t* status, int d, int j) {
  const double ang = double(d) * freq[j];                 // fp64 angle, as the table was built
  atomicOr(status, 2);
  return make_float2(float(cos(ang)), float(sin(ang)));
}

template <typename T, int NAX>
__device__ __forceinline__ void rotate_unit(const Geom& g, const int (&dl)[NAX], int j0, uint4& lo, uint4& hi) {
  constexpr int V = Elem<T>::kPerVec;
  float x[V], y[V];
  Elem<T>::unpack(lo, x);
  Elem<T>::unpack(hi, y);
  const int half = g.d >> 1;
  auto axis_delta = [&](int j) -> int {
    if (NAX == 1) return dl[0];
    return j < g.sec_t ? dl[0] : (j < g.sec_t + g.sec_h ? dl[NAX > 1 ? 1 : 0] : dl[NAX > 2 ? 2 : 0]);
  };
  const int d_first = axis_delta(j0), d_last = axis_delta(j0 + V - 1);
  if (d_first == d_last) {                                  // the whole unit belongs to one axis (the usual case)
    const int r = -d_first;
    if (r == 0) return;                                     // bit-exact copy
    if (r > 0 && r < g.table_rows) {
      const float4* tab = reinterpret_cast<const float4*>(g.rope_tab + size_t(r) * half + j0);
#pragma unroll
      for (int p = 0; p < V; p += 2) {
        const float4 cs = __ldg(tab + (p >> 1));            // (cos, sin) of pairs j0+p, j0+p+1
        rot_pair(x[p], y[p], cs.x, cs.y);
        rot_pair(x[p + 1], y[p + 1], cs.z, cs.w);
      }
    } else {
#pragma unroll
      for (int p = 0; p < V; ++p) {
        const float2 cs = slow_cos_sin(g.rope_freq, g.status, d_first, j0 + p);
        rot_pair(x[p], y[p], cs.x, cs.y);
      }
    }
  } else {                                                  // unit straddles two M-RoPE sections
#pragma unroll
    for (int p = 0; p < V; ++p) {
      const int d = axis_delta(j0 + p), r = -d;
      if (r != 0) {
        const float2 cs = (r > 0 && r < g.table_rows) ? __ldg(&g.rope_tab[size_t(r) * half + j0 + p])
                                                       : slow_cos_sin(g.rope_freq, g.status, d, j0 + p);
        rot_pair(x[p], y[p], cs.x, cs.y);
      }
    }
  }
  lo = Elem<T>::pack(x);
  hi = Elem<T>::pack(y);
}

// grid = (blocks per slab, B*L); each thread walks units idx, idx + stride, ... of its (stream, layer).
// kMode: kGatherKV moves K and V; kGatherK only K (V's compaction is deferred into the next update's scoring
// kernel, see tc_v_mover in k_score_tc.cuh); kGatherV only V (flush of a deferred compaction).
constexpr int kGatherKV = 0, kGatherK = 1, kGatherV = 2;

template <typename T, int NAX, int kMode>
__global__ void __launch_bounds__(kGatherThreads, 4)
k_gather(Geom g, int cur) {
  pdl_wait();
  pdl_launch_dependents();
  constexpr int V = Elem<T>::kPerVec;
  const int bl = blockIdx.y;
  const int half = g.d >> 1;
  const int uph = half / V;                                 // units per head
  const int upr = g.Hkv * uph;                              // units per token row
  const int total = layer_keep(g, bl % g.L) * upr;      // rows this layer holds after the update (its budget, or all of them)
  const size_t slab_src = size_t(bl) * 2 + cur, slab_dst = size_t(bl) * 2 + (cur ^ 1);
  const T* ks = reinterpret_cast<const T*>(g.kc) + slab_src * g.cap * g.row_elems;
  const T* vs = reinterpret_cast<const T*>(g.vc) + slab_src * g.cap * g.row_elems;
  T* kd = reinterpret_cast<T*>(g.kc) + slab_dst * g.cap * g.row_elems;
  T* vd = reinterpret_cast<T*>(g.vc) + slab_dst * g.cap * g.row_elems;
  const int32_t* kept = g.kept + size_t(bl) * g.budget;
  const int32_t* delta = g.delta + size_t(bl) * g.n_axes * g.budget;   // written by k_select

  // One unit per thread and trip (K-only mode with 2-4 units per trip, or with 5-6 blocks per SM, measured slower: 81-99 us
  // against 72 us -- register spills at 64 registers, fewer resident blocks above that).  A thread's unit index advances by
  // `stride` per trip; its (row, unit in row) pair advances by (stride / upr, stride % upr) with a carry -- no integer
  // division inside the loop (each costs ~25 instructions and a MUFU.RCP round trip in the dependent chain of the next loads).
  const int rows = total / upr;
  const int stride = gridDim.x * kGatherThreads;
  const int ds = stride / upr, du = stride - ds * upr;
  const int sh = __ffs(uph) - 1;                            // uph = (d / 2) / V is a power of two (d is 32, 64 or 128)
  int idx = blockIdx.x * kGatherThreads + threadIdx.x;
  if (idx >= total) return;
  int s = idx / upr, u = idx - s * upr;
  int src = __ldcg(kept + s), dl[NAX];
#pragma unroll
  for (int a = 0; a < NAX; ++a) dl[a] = __ldcg(delta + a * g.budget + s);

#pragma unroll 1
  while (true) {
    const int j0 = (u & (uph - 1)) * V, e = (u >> sh) * g.d + j0;
    const size_t so = size_t(max(src, 0)) * g.row_elems + e;   // src < 0: the summary-token slot, written by k_summary
    uint4 klo, khi, vlo, vhi;
    klo = khi = vlo = vhi = make_uint4(0, 0, 0, 0);
    if (kMode != kGatherV) { klo = ldg_stream(ks + so); khi = ldg_stream(ks + so + half); }
    if (kMode != kGatherK) { vlo = ldg_stream(vs + so); vhi = ldg_stream(vs + so + half); }
    // the next trip's position, row index and deltas (prefetched while this trip's vectors are in flight)
    const int idx_n = idx + stride;
    int s_n = s + ds, u_n = u + du;
    if (u_n >= upr) { u_n -= upr; ++s_n; }
    const int s_ld = min(s_n, rows - 1);
    const int src_n = __ldcg(kept + s_ld);
    int dl_n[NAX];
#pragma unroll
    for (int a = 0; a < NAX; ++a) dl_n[a] = __ldcg(delta + a * g.budget + s_ld);

    bool any = false;
#pragma unroll
    for (int a = 0; a < NAX; ++a) any |= dl[a] != 0;
    if (kMode != kGatherV && any) rotate_unit<T, NAX>(g, dl, j0, klo, khi);
    const size_t dof = size_t(s) * g.row_elems + e;
    if (src >= 0) {
      if (kMode != kGatherV) { stg_stream(kd + dof, klo); stg_stream(kd + dof + half, khi); }
      if (kMode != kGatherK) { stg_stream(vd + dof, vlo); stg_stream(vd + dof + half, vhi); }
    }
    if (idx_n >= total) break;
    idx = idx_n; s = s_n; u = u_n; src = src_n;
#pragma unroll
    for (int a = 0; a < NAX; ++a) dl[a] = dl_n[a];
  }
}

}  // namespace hk
