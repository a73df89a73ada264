// a5 + a7 fused -- gather-compaction K_l[I_l], V_l[I_l] (Eq. 6) with the delta rotary
// correction of the kept keys (Eq. 9-10; M-RoPE Eq. 12-13), from the
// current buffer into the other one.  HBM-bound: every thread moves 4 x 16 bytes (K lo/hi halves of a
// rotary pair group + the same two vectors of V), 128-bit coalesced, streaming cache policy.
//
// A "unit" = kPerVec rotary pairs of one KV head: elements [j0, j0+kPerVec) and [j0+d/2, ...) of the head.
// Rotation: angle table (cos, sin)(delta * theta_j) built in fp64 at create time; fp32 products and
// sums WITHOUT fused multiply-add, round-to-nearest-even to the storage dtype; delta = 0 is a bit-exact
// copy (DESIGN c14).  Deltas outside the table take an fp64 sincos slow path (status bit 1).
#pragma once
#include "common.cuh"

namespace hk {

constexpr int kGatherThreads = 256;

struct UnitCoord { int s, head, k; };

template <typename T>
__device__ inline void rotate_unit(const Geom& g, const int* dl, int j0, uint4& lo, uint4& hi) {
  constexpr int V = Elem<T>::kPerVec;
  float x[V], y[V];
  Elem<T>::unpack(lo, x);
  Elem<T>::unpack(hi, y);
  const int half = g.d >> 1;
#pragma unroll
  for (int p = 0; p < V; ++p) {
    const int j = j0 + p;
    const int a = (g.n_axes == 1) ? 0 : (j >= g.sec_t) + (j >= g.sec_t + g.sec_h);
    const int d = dl[a];
    if (d != 0) {
      float c, s;
      const int r = -d;
      if (r > 0 && r < g.table_rows) {
        const float2 cs = __ldg(&g.rope_tab[size_t(r) * half + j]);
        c = cs.x; s = cs.y;
      } else {                                          // outside the table: fp64 angle, as the table was built
        const double ang = double(d) * g.rope_freq[j];
        c = float(cos(ang)); s = float(sin(ang));
        atomicOr(g.status, 2);
      }
      const float xn = __fsub_rn(__fmul_rn(x[p], c), __fmul_rn(y[p], s));
      const float yn = __fadd_rn(__fmul_rn(x[p], s), __fmul_rn(y[p], c));
      x[p] = xn; y[p] = yn;
    }
  }
  lo = Elem<T>::pack(x);
  hi = Elem<T>::pack(y);
}

template <typename T>
__global__ void __launch_bounds__(kGatherThreads)
k_gather(Geom g, int cur) {
  constexpr int V = Elem<T>::kPerVec;
  const int bl = blockIdx.y;
  const int half = g.d >> 1;
  const int uph = half / V;                             // units per head
  const int upr = g.Hkv * uph;                          // units per token row
  const int total = g.budget * upr;
  const size_t slab_src = size_t(bl) * 2 + cur, slab_dst = size_t(bl) * 2 + (cur ^ 1);
  const T* ks = reinterpret_cast<const T*>(g.kc) + slab_src * g.cap * g.row_elems;
  const T* vs = reinterpret_cast<const T*>(g.vc) + slab_src * g.cap * g.row_elems;
  T* kd = reinterpret_cast<T*>(g.kc) + slab_dst * g.cap * g.row_elems;
  T* vd = reinterpret_cast<T*>(g.vc) + slab_dst * g.cap * g.row_elems;
  const int32_t* kept = g.kept + size_t(bl) * g.budget;
  const int32_t* pos_old = g.posc + slab_src * g.n_axes * g.cap;
  const int32_t* pos_new = g.posc + slab_dst * g.n_axes * g.cap;   // written by k_select

  const int stride = gridDim.x * kGatherThreads;
  for (int idx = blockIdx.x * kGatherThreads + threadIdx.x; idx < total; idx += 2 * stride) {
    // two independent units per iteration -> 8 x 16-byte loads in flight per thread
    const int idx2 = idx + stride;
    const bool two = idx2 < total;
    const int s0 = idx / upr, u0 = idx % upr;
    const int s1 = two ? idx2 / upr : s0, u1 = two ? idx2 % upr : u0;
    const int src0 = __ldg(kept + s0), src1 = __ldg(kept + s1);
    const int e0 = (u0 / uph) * g.d + (u0 % uph) * V, e1 = (u1 / uph) * g.d + (u1 % uph) * V;
    const size_t so0 = size_t(src0) * g.row_elems + e0, so1 = size_t(src1) * g.row_elems + e1;
    uint4 klo0 = ldg_stream(ks + so0), khi0 = ldg_stream(ks + so0 + half);
    uint4 vlo0 = ldg_stream(vs + so0), vhi0 = ldg_stream(vs + so0 + half);
    uint4 klo1, khi1, vlo1, vhi1;
    if (two) {
      klo1 = ldg_stream(ks + so1); khi1 = ldg_stream(ks + so1 + half);
      vlo1 = ldg_stream(vs + so1); vhi1 = ldg_stream(vs + so1 + half);
    }
    int dl0[3] = {0, 0, 0}, dl1[3] = {0, 0, 0};
    for (int a = 0; a < g.n_axes; ++a) {
      dl0[a] = __ldg(pos_new + size_t(a) * g.cap + s0) - __ldg(pos_old + size_t(a) * g.cap + src0);
      dl1[a] = __ldg(pos_new + size_t(a) * g.cap + s1) - __ldg(pos_old + size_t(a) * g.cap + src1);
    }
    if (dl0[0] | dl0[1] | dl0[2]) rotate_unit<T>(g, dl0, (u0 % uph) * V, klo0, khi0);
    const size_t do0 = size_t(s0) * g.row_elems + e0;
    stg_stream(kd + do0, klo0); stg_stream(kd + do0 + half, khi0);
    stg_stream(vd + do0, vlo0); stg_stream(vd + do0 + half, vhi0);
    if (two) {
      if (dl1[0] | dl1[1] | dl1[2]) rotate_unit<T>(g, dl1, (u1 % uph) * V, klo1, khi1);
      const size_t do1 = size_t(s1) * g.row_elems + e1;
      stg_stream(kd + do1, klo1); stg_stream(kd + do1 + half, khi1);
      stg_stream(vd + do1, vlo1); stg_stream(vd + do1 + half, vhi1);
    }
  }
}

}  // namespace hk
