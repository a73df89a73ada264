// f1 -- summary token of the evicted tokens of every deep layer (Alg. 1):
//   v_sum = Mean(V_p);  k_sum = Mean(ApplyDelta(K_p, RotaryDelta(P_p -> t))),  t = pos_offset + budget - 1 at a re-index
//   step, the position after the newest token between the re-index steps of the lazy mode (DESIGN f1),
// written to slot budget-1 of the NEW buffer (k_gather leaves that slot alone; k_select set its position).
// One block per (KV head, stream x deep layer): thread = (rotary pair j, token lane q); token lane q walks the
// evicted tokens q, q + kSumLanes, ...  (cos, sin) from a table built in fp64 at create time for every delta in
// the table range (fp64 sincos otherwise), rotation in fp32 without FMA exactly as in k_gather, sums in fp64, lanes reduced
// in shared memory in fixed order, one rounding to the storage dtype.  ~E x 2 KB per layer: latency only.
#pragma once
#include "common.cuh"

namespace hk {

constexpr int kSumLanes = 16;

template <typename T>
__global__ void __launch_bounds__(64 * kSumLanes)
k_summary(Geom g, int cur, int Tn, int t, int reindex) {
  __shared__ double red[kSumLanes][4][64];                 // [token lane][kx, ky, vx, vy][pair]
  extern __shared__ int s_list[];                          // [2][n_ev]: source row, rotary delta of every evicted token
  pdl_wait();
  pdl_launch_dependents();
  const int half = g.d >> 1;
  const int j = threadIdx.x % 64, q = threadIdx.x / 64;    // blockDim.x = 64 * kSumLanes; pairs j, j + 64 if half > 64
  const int kvh = blockIdx.x;
  const int b = blockIdx.y / g.n_deep, l = g.L - g.n_deep + blockIdx.y % g.n_deep;
  const int bl = b * g.L + l;
  // layer-dependent budgets (DESIGN f1 x f4): this layer's own candidates and budget; a layer still under its budget at this
  // arrival evicts nothing and makes no summary token
  Tn = layer_T(g, l, Tn);
  if (layer_keep(g, l) >= Tn) return;
  const int n_keep = layer_keep(g, l) - 1, n_ev = Tn - n_keep;
  if (reindex) t = g.pos_offset + n_keep;               // the next contiguous position (Alg. 1 step 3)
  const size_t slab_src = size_t(bl) * 2 + cur, slab_dst = size_t(bl) * 2 + (cur ^ 1);
  const T* ks = reinterpret_cast<const T*>(g.kc) + slab_src * g.cap * g.row_elems + kvh * g.d;
  const T* vs = reinterpret_cast<const T*>(g.vc) + slab_src * g.cap * g.row_elems + kvh * g.d;
  const int32_t* pos_old = g.posc + slab_src * g.cap;      // 1D RoPE only (validated at create)
  const int32_t* ev = g.evicted + size_t(bl) * g.n_evict_max;
  int* s_src = s_list;
  int* s_dl = s_list + n_ev;
  for (int i = threadIdx.x; i < n_ev; i += blockDim.x) {   // one dependent-load chain per token, all in flight at once
    const int src = __ldcg(ev + i);
    s_src[i] = src; s_dl[i] = t - __ldcg(pos_old + src);
  }
  __syncthreads();
  for (int j0 = 0; j0 < half; j0 += 64) {
    const int jj = j0 + j;
    double kx = 0.0, ky = 0.0, vx = 0.0, vy = 0.0;
    if (jj < half) {
#pragma unroll 4
      for (int i = q; i < n_ev; i += kSumLanes) {
        const int src = s_src[i];
        const int delta = s_dl[i];
        const int r = delta + g.sum_tab_zero;
        float c, s;
        if (r >= 0 && r < g.sum_tab_rows) { const float2 cs = __ldg(g.sum_tab + size_t(r) * half + jj); c = cs.x; s = cs.y; }
        else { const double ang = double(delta) * g.rope_freq[jj]; c = float(cos(ang)); s = float(sin(ang)); }   // explicit pos_start jumps
        const size_t o = size_t(src) * g.row_elems;
        const float x = Elem<T>::to_float(__ldcg(ks + o + jj)), y = Elem<T>::to_float(__ldcg(ks + o + jj + half));
        float xr = x, yr = y;
        if (delta != 0) {
          xr = __fsub_rn(__fmul_rn(x, c), __fmul_rn(y, s));
          yr = __fadd_rn(__fmul_rn(x, s), __fmul_rn(y, c));
        }
        kx += double(xr); ky += double(yr);
        vx += double(Elem<T>::to_float(__ldcg(vs + o + jj))); vy += double(Elem<T>::to_float(__ldcg(vs + o + jj + half)));
      }
    }
    __syncthreads();
    red[q][0][j] = kx; red[q][1][j] = ky; red[q][2][j] = vx; red[q][3][j] = vy;
    __syncthreads();
    if (q == 0 && jj < half) {
      double s4[4] = {0.0, 0.0, 0.0, 0.0};
      for (int w = 0; w < kSumLanes; ++w)
        for (int c = 0; c < 4; ++c) s4[c] += red[w][c][j];
      const double inv = 1.0 / double(n_ev);
      T* kd = reinterpret_cast<T*>(g.kc) + (slab_dst * g.cap + n_keep) * g.row_elems + kvh * g.d;
      T* vd = reinterpret_cast<T*>(g.vc) + (slab_dst * g.cap + n_keep) * g.row_elems + kvh * g.d;
      kd[jj] = T(float(s4[0] * inv)); kd[jj + half] = T(float(s4[1] * inv));
      vd[jj] = T(float(s4[2] * inv)); vd[jj + half] = T(float(s4[3] * inv));
    }
  }
}

}  // namespace hk
