// a1 -- attention importance W (Eq. 2) on the 5th-gen tensor cores: bf16, head_dim 128.
//
// Same two-pass recompute as the CUDA-core path (k_score_simt.cuh), but each pass is a persistent,
// warp-specialised tcgen05 kernel fed by TMA, with fp32 accumulators in TMEM:
//   pass 1 k_tc_stats  : D[row, tok] = Q_blk K_tile^T, probe rows on TMEM lanes -> each thread owns one
//                        probe row and keeps its running (max, sum exp2) over the tokens: no cross-lane work.
//   combine            : per probe row c_r = m_r + log2 Z_r.
//   pass 2 k_tc_colsum : D[tok, row] = K_tile Q^T, tokens on TMEM lanes -> each thread owns one token and
//                        accumulates sum_r exp2(s * scale - c_r): again no cross-lane work.
// A "group" = (stream, scored layer, KV head, row super-chunk of <= 512 probe rows); its Q rows stay in
// shared memory while the K tiles of the group stream through a TMA ring.  The flattened (group, tile)
// space is cut into equal contiguous ranges, one per CTA (<= #SM CTAs, 1 CTA/SM).
#pragma once
#include "host_state.cuh"
#include "tc_ptx.cuh"

namespace hk {

constexpr int kTcRowsMax = 512;                 // probe rows resident per group (Q tile = 128 KB)
constexpr int kTcQHalfBytes = kTcRowsMax * 128; // one 64-column half of the Q tile
constexpr int kTcKBytes = 64 * 1024;            // K ring: 4 x 16 KB (pass 1) or 2 x 32 KB (pass 2)
constexpr int kTcSmemBytes = 2 * kTcQHalfBytes + kTcKBytes + kTcRowsMax * 4 + 512 + 1024;
constexpr int kTcStatsThreads = 64 + 8 * 32;    // producer, MMA, 8 epilogue warps
constexpr int kTcColsumThreads = 64 + 8 * 32;   // producer, MMA, 8 epilogue warps
constexpr int kTcSegTiles = 8;                  // pass 1: 64-token tiles per segment (one partial per segment,
                                                // so the merge order never depends on the CTA schedule)

struct TcArgs {
  Geom g;
  int cur, Tn, P;
  float scale_log2;
  int R, RS, n_sc;          // probe rows per KV head (G*P), rows per super-chunk, super-chunks per KV head
  int tpg;                  // token tiles per group (64-token tiles in pass 1, 128-token tiles in pass 2)
  int n_groups;             // B * Ls * Hkv * n_sc
  int spg;                  // pass 1: 512-token segments per group = partial (m, z) slots per probe row
};

// ---- schedule: CTA c owns flattened units [c*U/nC, (c+1)*U/nC) -----------------------------------
__host__ __device__ inline long long tc_unit_begin(long long U, int n_cta, int c) { return (U * c) / n_cta; }
__host__ __device__ inline int tc_cta_of_unit(long long U, int n_cta, long long u) { return int(((u + 1) * n_cta - 1) / U); }

struct TcGroup { int bl, kvh, sc, rs_valid, stat_row0; long long q_row0; };
__device__ inline TcGroup tc_group(const TcArgs& a, int gi) {
  TcGroup r;
  const Geom& g = a.g;
  const int Ls = g.L - g.n_shallow;
  r.sc = gi % a.n_sc;
  r.kvh = (gi / a.n_sc) % g.Hkv;
  const int bls = gi / (a.n_sc * g.Hkv);
  r.bl = (bls / Ls) * g.L + g.n_shallow + bls % Ls;
  r.rs_valid = min(a.RS, a.R - r.sc * a.RS);
  r.stat_row0 = r.kvh * a.R + r.sc * a.RS;
  r.q_row0 = (long long)r.bl * g.Hq * a.P + r.stat_row0;
  return r;
}

struct TcSmem {
  uint8_t* q;        // [2 halves][512 rows][128 B], 128B-swizzled
  uint8_t* k;        // K ring
  float* c;          // [512] per-row c_r (pass 2)
  uint64_t* bars;    // mbarriers
  uint32_t* tmem;    // TMEM base address written by tcgen05.alloc
};
__device__ inline TcSmem tc_carve(uint8_t* raw) {
  uint8_t* p = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(raw) + 1023) & ~uintptr_t(1023));
  TcSmem s;
  s.q = p; p += 2 * kTcQHalfBytes;
  s.k = p; p += kTcKBytes;
  s.c = reinterpret_cast<float*>(p); p += kTcRowsMax * 4;
  s.bars = reinterpret_cast<uint64_t*>(p); p += 256;
  s.tmem = reinterpret_cast<uint32_t*>(p);
  return s;
}

// Loads the group's Q rows (both 64-column halves) in 64-row boxes.
__device__ inline void tc_load_q(const TcSmem& s, const CUtensorMap* tq, uint64_t* bar, const TcGroup& gr) {
  const int n_box = (gr.rs_valid + 63) / 64;
  ptx::mbar_expect_tx(bar, uint32_t(n_box) * 2 * 8192);
  for (int h = 0; h < 2; ++h)
    for (int bx = 0; bx < n_box; ++bx)
      ptx::tma_load_2d(s.q + h * kTcQHalfBytes + bx * 8192, tq, bar, h * 64, int(gr.q_row0) + bx * 64);
}

// =====================================================================================================
// pass 1: per probe row, partial (max, sum exp2) over this CTA's token range of the group
// =====================================================================================================
__global__ void __launch_bounds__(kTcStatsThreads, 1)
k_tc_stats(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k, TcArgs a) {
  extern __shared__ uint8_t smem_raw[];
  const TcSmem s = tc_carve(smem_raw);
  constexpr int NS = 4, TN = 64, KSTAGE = 16384;
  uint64_t* k_full = s.bars;            // [NS]
  uint64_t* k_empty = s.bars + NS;      // [NS]
  uint64_t* t_full = s.bars + 2 * NS;   // [2]
  uint64_t* t_empty = t_full + 2;       // [2]
  uint64_t* q_full = t_empty + 2;
  uint64_t* q_empty = q_full + 1;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long U = (long long)a.n_groups * a.spg;                     // schedule unit = (group, segment)
  const int n_cta = gridDim.x, cta = blockIdx.x;
  const long long s0 = tc_unit_begin(U, n_cta, cta), s1 = tc_unit_begin(U, n_cta, cta + 1);

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmap_q); ptx::prefetch_tmap(&tmap_k);
    for (int i = 0; i < NS; ++i) { ptx::mbar_init(&k_full[i], 1); ptx::mbar_init(&k_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&t_full[i], 1); ptx::mbar_init(&t_empty[i], 8); }
    ptx::mbar_init(q_full, 1); ptx::mbar_init(q_empty, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc(s.tmem, 512);
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *s.tmem;

  if (warp == 0) {
    // ---------------- TMA producer ----------------
    if (lane == 0) {
      int ks = 0, kph = 0, n_q = 0, prev = -1;
      for (long long u = s0; u < s1; ++u) {
        const int gi = int(u / a.spg), sg = int(u % a.spg);
        const TcGroup gr = tc_group(a, gi);
        if (gi != prev) {
          if (n_q > 0) ptx::mbar_wait(q_empty, (n_q - 1) & 1);
          tc_load_q(s, &tmap_q, q_full, gr);
          ++n_q; prev = gi;
        }
        const int t_end = min(a.tpg, (sg + 1) * kTcSegTiles);
        for (int t = sg * kTcSegTiles; t < t_end; ++t) {
          ptx::mbar_wait(&k_empty[ks], kph ^ 1);
          ptx::mbar_expect_tx(&k_full[ks], KSTAGE);
          const int row = int((size_t(gr.bl) * 2 + a.cur) * a.g.cap) + t * TN;
          for (int h = 0; h < 2; ++h)
            ptx::tma_load_2d(s.k + ks * KSTAGE + h * 8192, &tmap_k, &k_full[ks], gr.kvh * 128 + h * 64, row);
          if (++ks == NS) { ks = 0; kph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ---------------- MMA issuer ----------------
    const uint32_t idesc = ptx::idesc_bf16_f32(128, TN);
    int ks = 0, kph = 0, as = 0, aph = 0, n_q = 0, prev = -1, n_rb = 0;
    for (long long u = s0; u < s1; ++u) {
      const int gi = int(u / a.spg), sg = int(u % a.spg);
      if (gi != prev) {
        const TcGroup gr = tc_group(a, gi);
        n_rb = (gr.rs_valid + 127) / 128;
        ptx::mbar_wait(q_full, n_q & 1);
        ++n_q; prev = gi;
      }
      const bool last_seg_of_group = (u + 1 == s1) || int((u + 1) / a.spg) != gi;
      const int t_end = min(a.tpg, (sg + 1) * kTcSegTiles);
      for (int t = sg * kTcSegTiles; t < t_end; ++t) {
        ptx::mbar_wait(&k_full[ks], kph);
        ptx::mbar_wait(&t_empty[as], aph ^ 1);
        ptx::tc_fence_after();
        if (lane == 0) {
          for (int rb = 0; rb < n_rb; ++rb) {
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
              const int h = kk >> 2;
              const uint64_t ad = ptx::smem_desc_sw128(ptx::smem_u32(s.q + h * kTcQHalfBytes + rb * 16384)) + uint64_t((kk & 3) * 2);
              const uint64_t bd = ptx::smem_desc_sw128(ptx::smem_u32(s.k + ks * KSTAGE + h * 8192)) + uint64_t((kk & 3) * 2);
              ptx::mma_bf16(tmem_base + as * 256 + rb * TN, ad, bd, idesc, kk > 0);
            }
          }
          ptx::mma_commit(&k_empty[ks]);
          ptx::mma_commit(&t_full[as]);
          if (last_seg_of_group && t + 1 == t_end) ptx::mma_commit(q_empty);
        }
        __syncwarp();
        if (++ks == NS) { ks = 0; kph ^= 1; }
        if (++as == 2) { as = 0; aph ^= 1; }
      }
    }
  } else {
    // ---------------- epilogue: two probe rows per thread (row blocks rb0, rb0+1), software-pipelined:
    // the TMEM load of one row block is always in flight while the other goes through the MUFU pipe ----
    const int e = warp - 2, rb0 = (e >> 2) * 2, lg = warp & 3;
    int as = 0, aph = 0;
    float m_run[2] = {-INFINITY, -INFINITY}, z[2] = {0.f, 0.f};
    float vA[TN], vB[TN];
    // running (max, sum exp2) of one row over one 64-token tile
    auto fold = [&](float (&v)[TN], int t, float& m_r, float& z_r) {
      const int n_valid = min(TN, a.Tn - t * TN);                       // ragged last tile of the group
      if (n_valid < TN) {
#pragma unroll
        for (int j = 0; j < TN; ++j) if (j >= n_valid) v[j] = -INFINITY;
      }
      float mx[4] = {v[0], v[1], v[2], v[3]};
#pragma unroll
      for (int j = 4; j < TN; j += 4) {
        mx[0] = fmaxf(mx[0], v[j]); mx[1] = fmaxf(mx[1], v[j + 1]);
        mx[2] = fmaxf(mx[2], v[j + 2]); mx[3] = fmaxf(mx[3], v[j + 3]);
      }
      const float m_new = fmaxf(m_r, fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * a.scale_log2);
#pragma unroll
      for (int j = 0; j < TN; ++j) v[j] = fmaf(v[j], a.scale_log2, -m_new);
#pragma unroll
      for (int j = 0; j < TN; ++j) v[j] = fast_exp2(v[j]);
      float sm[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int j = 0; j < TN; j += 4) { sm[0] += v[j]; sm[1] += v[j + 1]; sm[2] += v[j + 2]; sm[3] += v[j + 3]; }
      z_r = z_r * fast_exp2(m_r - m_new) + ((sm[0] + sm[1]) + (sm[2] + sm[3]));
      m_r = m_new;
    };
    long long u = s0;
    if (u < s1) {
      int gi = int(u / a.spg), sg = int(u % a.spg);
      TcGroup gr = tc_group(a, gi);
      int t = sg * kTcSegTiles, t_end = min(a.tpg, t + kTcSegTiles);
      bool act0 = rb0 * 128 + lg * 32 < gr.rs_valid, act1 = (rb0 + 1) * 128 + lg * 32 < gr.rs_valid;
      const uint32_t lane_base = uint32_t(lg * 32) << 16;
      ptx::mbar_wait(&t_full[as], aph);
      ptx::tc_fence_after();
      if (act0) { ptx::tmem_ld32(tmem_base + lane_base + as * 256 + rb0 * TN, vA); ptx::tmem_ld32(tmem_base + lane_base + as * 256 + rb0 * TN + 32, vA + 32); }
      while (true) {
        ptx::tmem_ld_wait();                                             // row block rb0 of tile t is in registers
        if (act1) { ptx::tmem_ld32(tmem_base + lane_base + as * 256 + (rb0 + 1) * TN, vB); ptx::tmem_ld32(tmem_base + lane_base + as * 256 + (rb0 + 1) * TN + 32, vB + 32); }
        if (act0) fold(vA, t, m_run[0], z[0]);
        ptx::tmem_ld_wait();                                             // row block rb0+1 too: free the TMEM stage
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&t_empty[as]);
        if (++as == 2) { as = 0; aph ^= 1; }
        // advance to the next tile of this CTA's range and start its first load
        const int t_cur = t, sg_cur = sg;
        const TcGroup gr_cur = gr;
        const bool seg_done = t + 1 >= t_end, act1_cur = act1;
        bool more = true;
        if (!seg_done) { ++t; }
        else if (++u < s1) {
          const int gi_n = int(u / a.spg);
          sg = int(u % a.spg);
          if (gi_n != gi) { gi = gi_n; gr = tc_group(a, gi); }
          t = sg * kTcSegTiles; t_end = min(a.tpg, t + kTcSegTiles);
        } else more = false;
        const bool act0_cur = act0;
        if (more) {
          act0 = rb0 * 128 + lg * 32 < gr.rs_valid; act1 = (rb0 + 1) * 128 + lg * 32 < gr.rs_valid;
          ptx::mbar_wait(&t_full[as], aph);
          ptx::tc_fence_after();
          if (act0) { ptx::tmem_ld32(tmem_base + lane_base + as * 256 + rb0 * TN, vA); ptx::tmem_ld32(tmem_base + lane_base + as * 256 + rb0 * TN + 32, vA + 32); }
        }
        if (act1_cur) fold(vB, t_cur, m_run[1], z[1]);
        if (seg_done) {                                                  // one partial per (row, segment)
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            const int row = (rb0 + k) * 128 + lg * 32 + lane;
            if ((k == 0 ? act0_cur : act1_cur) && row < gr_cur.rs_valid) {
              float* out = a.g.partial + ((size_t(gr_cur.bl) * a.g.Hq * a.g.p_max + gr_cur.stat_row0 + row) * a.spg + sg_cur) * 2;
              out[0] = m_run[k]; out[1] = z[k];
            }
            m_run[k] = -INFINITY; z[k] = 0.f;
          }
        }
        if (!more) break;
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) ptx::tmem_dealloc(tmem_base, 512);
}

// =====================================================================================================
// pass 2: per token, sum over the group's probe rows of exp2(s * scale - c_r)
// =====================================================================================================
__global__ void __launch_bounds__(kTcColsumThreads, 1)
k_tc_colsum(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k, TcArgs a) {
  extern __shared__ uint8_t smem_raw[];
  const TcSmem s = tc_carve(smem_raw);
  constexpr int NS = 2, TN = 128, KSTAGE = 32768;
  __shared__ float acc_x[2][128];       // partial sums of the upper column-half warps (double-buffered)
  uint64_t* k_full = s.bars;            // [NS]
  uint64_t* k_empty = s.bars + NS;      // [NS]
  uint64_t* t_full = s.bars + 2 * NS;   // [2]
  uint64_t* t_empty = t_full + 2;       // [2]
  uint64_t* q_full = t_empty + 2;
  uint64_t* q_empty = q_full + 1;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long U = (long long)a.n_groups * a.tpg;
  const int n_cta = gridDim.x, cta = blockIdx.x;
  const long long u0 = tc_unit_begin(U, n_cta, cta), u1 = tc_unit_begin(U, n_cta, cta + 1);

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmap_q); ptx::prefetch_tmap(&tmap_k);
    for (int i = 0; i < NS; ++i) { ptx::mbar_init(&k_full[i], 1); ptx::mbar_init(&k_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&t_full[i], 1); ptx::mbar_init(&t_empty[i], 8); }
    ptx::mbar_init(q_full, 1); ptx::mbar_init(q_empty, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc(s.tmem, 512);
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *s.tmem;

  if (warp == 0) {
    if (lane == 0) {
      int ks = 0, kph = 0, n_q = 0, prev = -1;
      for (long long u = u0; u < u1; ++u) {
        const int gi = int(u / a.tpg), t = int(u % a.tpg);
        const TcGroup gr = tc_group(a, gi);
        if (gi != prev) {
          if (n_q > 0) ptx::mbar_wait(q_empty, (n_q - 1) & 1);
          tc_load_q(s, &tmap_q, q_full, gr);
          ++n_q; prev = gi;
        }
        ptx::mbar_wait(&k_empty[ks], kph ^ 1);
        ptx::mbar_expect_tx(&k_full[ks], KSTAGE);
        const int row = int((size_t(gr.bl) * 2 + a.cur) * a.g.cap) + t * TN;
        for (int h = 0; h < 2; ++h)
          for (int bx = 0; bx < 2; ++bx)
            ptx::tma_load_2d(s.k + ks * KSTAGE + h * 16384 + bx * 8192, &tmap_k, &k_full[ks], gr.kvh * 128 + h * 64, row + bx * 64);
        if (++ks == NS) { ks = 0; kph ^= 1; }
      }
    }
  } else if (warp == 1) {
    int ks = 0, kph = 0, as = 0, aph = 0, n_q = 0, prev = -1, rs32 = 0;
    for (long long u = u0; u < u1; ++u) {
      const int gi = int(u / a.tpg);
      if (gi != prev) {
        const TcGroup gr = tc_group(a, gi);
        rs32 = (gr.rs_valid + 31) & ~31;
        ptx::mbar_wait(q_full, n_q & 1);
        ++n_q; prev = gi;
      }
      ptx::mbar_wait(&k_full[ks], kph);
      for (int c0 = 0; c0 < rs32; c0 += 256) {                           // probe-row chunks of <= 256 columns
        const int nc = min(256, rs32 - c0);
        ptx::mbar_wait(&t_empty[as], aph ^ 1);
        ptx::tc_fence_after();
        if (lane == 0) {
          const uint32_t idesc = ptx::idesc_bf16_f32(128, nc);
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const int h = kk >> 2;
            const uint64_t ad = ptx::smem_desc_sw128(ptx::smem_u32(s.k + ks * KSTAGE + h * 16384)) + uint64_t((kk & 3) * 2);
            const uint64_t bd = ptx::smem_desc_sw128(ptx::smem_u32(s.q + h * kTcQHalfBytes + c0 * 128)) + uint64_t((kk & 3) * 2);
            ptx::mma_bf16(tmem_base + as * 256, ad, bd, idesc, kk > 0);
          }
          ptx::mma_commit(&t_full[as]);
        }
        __syncwarp();
        if (++as == 2) { as = 0; aph ^= 1; }
      }
      if (lane == 0) {
        ptx::mma_commit(&k_empty[ks]);
        const bool last_of_group = (u + 1 == u1) || int((u + 1) / a.tpg) != gi;
        if (last_of_group) ptx::mma_commit(q_empty);
      }
      __syncwarp();
      if (++ks == NS) { ks = 0; kph ^= 1; }
    }
  } else {
    // ---------------- epilogue: one token per thread, two warps (column halves) per 32-lane quarter ----
    const int e = warp - 2, half = e >> 2, lg = warp & 3;
    const int tok_in_tile = lg * 32 + lane;
    const int et = threadIdx.x - 64;                                     // 0..255
    int as = 0, aph = 0, prev = -1, rs32 = 0;
    TcGroup gr{};
    for (long long u = u0; u < u1; ++u) {
      const int gi = int(u / a.tpg), t = int(u % a.tpg);
      if (gi != prev) {
        gr = tc_group(a, gi); prev = gi;
        rs32 = (gr.rs_valid + 31) & ~31;
        ptx::named_bar_sync(1, 256);                                     // everyone is done with the old c_r
        // merge the row's per-segment (m, z) of pass 1 in segment order: c_r = m_r + log2 Z_r
        const float* pr = a.g.partial + (size_t(gr.bl) * a.g.Hq * a.g.p_max + gr.stat_row0) * a.spg * 2;
        for (int i = et; i < kTcRowsMax; i += 256) {
          float c = INFINITY;                                            // rows past the group: exp2(-inf) = 0
          if (i < gr.rs_valid) {
            const float2* p2 = reinterpret_cast<const float2*>(pr + size_t(i) * a.spg * 2);
            float m = -INFINITY;
            for (int j = 0; j < a.spg; ++j) m = fmaxf(m, p2[j].x);
            float z = 0.f;
            for (int j = 0; j < a.spg; ++j) z += p2[j].y * fast_exp2(p2[j].x - m);
            c = m + log2f(z);
          }
          s.c[i] = c;
        }
        ptx::named_bar_sync(1, 256);
      }
      float acc[4] = {0.f, 0.f, 0.f, 0.f};
      // 32 probe rows of this token: FFMA, MUFU and FADD phases kept apart so no warp waits on its own exp
      auto fold = [&](float (&v)[32], int col) {
        const float4* c4 = reinterpret_cast<const float4*>(s.c + col);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float4 c = c4[j];
          v[4 * j] = fmaf(v[4 * j], a.scale_log2, -c.x);
          v[4 * j + 1] = fmaf(v[4 * j + 1], a.scale_log2, -c.y);
          v[4 * j + 2] = fmaf(v[4 * j + 2], a.scale_log2, -c.z);
          v[4 * j + 3] = fmaf(v[4 * j + 3], a.scale_log2, -c.w);
        }
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = fast_exp2(v[j]);
#pragma unroll
        for (int j = 0; j < 32; j += 4) { acc[0] += v[j]; acc[1] += v[j + 1]; acc[2] += v[j + 2]; acc[3] += v[j + 3]; }
      };
      for (int c0 = 0; c0 < rs32; c0 += 256) {
        const int nc = min(256, rs32 - c0);
        ptx::mbar_wait(&t_full[as], aph);
        ptx::tc_fence_after();
        // this warp's 32-column blocks (every other one): the next block's TMEM load is in flight while
        // the current one goes through the MUFU pipe
        const uint32_t tbase = tmem_base + (uint32_t(lg * 32) << 16) + as * 256 + half * 32;
        const int nb = (nc - half * 32 + 63) / 64;
        float vA[32], vB[32];
        if (nb > 0) ptx::tmem_ld32(tbase, vA);
        for (int k = 0; k < nb; k += 2) {
          ptx::tmem_ld_wait();
          if (k + 1 < nb) ptx::tmem_ld32(tbase + (k + 1) * 64, vB);
          fold(vA, c0 + half * 32 + k * 64);
          if (k + 1 < nb) {
            ptx::tmem_ld_wait();
            if (k + 2 < nb) ptx::tmem_ld32(tbase + (k + 2) * 64, vA);
            fold(vB, c0 + half * 32 + (k + 1) * 64);
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&t_empty[as]);
        if (++as == 2) { as = 0; aph ^= 1; }
      }
      // merge the two column halves (one 64-thread barrier per lane quarter, double-buffered exchange)
      // and store W's per-(KV head, super-chunk) column sum of this token
      const float mine = (acc[0] + acc[1]) + (acc[2] + acc[3]);
      const int par = int(u & 1);
      if (half == 1) acc_x[par][tok_in_tile] = mine;
      ptx::named_bar_sync(2 + lg, 64);
      if (half == 0) {
        const int tok = t * TN + tok_in_tile;
        if (tok < a.Tn)
          a.g.colsum[(size_t(gr.bl) * a.g.n_vh_max + gr.kvh * a.n_sc + gr.sc) * a.g.cap + tok] = mine + acc_x[par][tok_in_tile];
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) ptx::tmem_dealloc(tmem_base, 512);
}

}  // namespace hk

// =====================================================================================================
// host side
// =====================================================================================================
namespace hk {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TcState {
  EncodeTiledFn encode = nullptr;
  CUtensorMap tmap_k;
  int n_sm = 0;
};

// 2D bf16 tensor map over [rows][cols] (cols contiguous), 64 x 64 boxes, 128-byte swizzle, zero OOB fill.
inline bool tc_make_map(TcState* st, CUtensorMap* out, const void* base, uint64_t cols, uint64_t rows) {
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {cols * 2};
  const cuuint32_t box[2] = {64, 64};
  const cuuint32_t estr[2] = {1, 1};
  return st->encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

inline bool tc_init(hermes_t* h) {
  const hermes_config& c = h->cfg;
  if (c.dtype != HERMES_BF16 || c.head_dim != 128) { h->err = "tcgen05 path needs bf16 and head_dim 128"; return false; }
  TcState* st = new (std::nothrow) TcState;
  if (!st) { h->err = "out of host memory"; return false; }
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    (void)cudaGetLastError();
    h->err = "cuTensorMapEncodeTiled not available from the driver";
    delete st; return false;
  }
  st->encode = reinterpret_cast<EncodeTiledFn>(fn);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, c.device) != cudaSuccess) { h->err = "cudaGetDeviceProperties failed"; delete st; return false; }
  st->n_sm = prop.multiProcessorCount;
  const Geom& g = h->geom;
  if (!tc_make_map(st, &st->tmap_k, g.kc, uint64_t(g.row_elems), uint64_t(g.B) * g.L * 2 * g.cap)) {
    h->err = "cuTensorMapEncodeTiled(K cache) failed"; delete st; return false;
  }
  if (cudaFuncSetAttribute(k_tc_stats, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemBytes) != cudaSuccess ||
      cudaFuncSetAttribute(k_tc_colsum, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemBytes) != cudaSuccess) {
    h->err = std::string("cudaFuncSetAttribute(tc kernels): ") + cudaGetErrorString(cudaGetLastError());
    delete st; return false;
  }
  h->tc_state = st;
  return true;
}

inline void tc_destroy(hermes_t* h) {
  delete static_cast<TcState*>(h->tc_state);
  h->tc_state = nullptr;
}

// Dense enough for the tensor pipe: at least one 32-row MMA column block and a few token tiles.
inline bool tc_profitable(const hermes_t* h, int Tn, int P) {
  return h->geom.G * P >= 32 && Tn >= 512;
}

struct TcProf {   // same event bracketing as hermes_api.cu's Prof, local to this header
  hermes_t* h; int id; cudaStream_t s;
  TcProf(hermes_t* h_, int id_, cudaStream_t s_) : h(h_), id(id_), s(s_) {
    if (h->profiling) { cudaEventRecord(h->timer.beg[id], s); h->timer.ran[id] = true; }
    ++h->last_launches;
  }
  ~TcProf() { if (h->profiling) cudaEventRecord(h->timer.end[id], s); }
};

inline int tc_score(hermes_t* h, const void* q_probe, int Tn, int P, float scale_log2, cudaStream_t s) {
  TcState* st = static_cast<TcState*>(h->tc_state);
  const Geom& g = h->geom;
  CUtensorMap tmap_q;
  if (!tc_make_map(st, &tmap_q, q_probe, 128, uint64_t(g.B) * g.L * g.Hq * P)) {
    h->err = "cuTensorMapEncodeTiled(Q_probe) failed (pointer must be 16-byte aligned)";
    return HERMES_EINVAL;
  }
  TcArgs a{};
  a.g = g; a.cur = h->cur; a.Tn = Tn; a.P = P; a.scale_log2 = scale_log2;
  a.R = g.G * P;
  a.n_sc = (a.R + kTcRowsMax - 1) / kTcRowsMax;
  a.RS = ((a.R + a.n_sc - 1) / a.n_sc + 31) & ~31;            // rows per super-chunk, multiple of 32
  a.n_sc = (a.R + a.RS - 1) / a.RS;
  a.n_groups = g.B * (g.L - g.n_shallow) * g.Hkv * a.n_sc;
  const int tpg1 = (Tn + 63) / 64, tpg2 = (Tn + 127) / 128;
  a.spg = (tpg1 + kTcSegTiles - 1) / kTcSegTiles;
  const long long U1 = (long long)a.n_groups * a.spg, U2 = (long long)a.n_groups * tpg2;
  const int n_cta1 = int(std::min<long long>(st->n_sm, U1)), n_cta2 = int(std::min<long long>(st->n_sm, U2));
  if (a.spg > h->lay.n_part_max || g.Hkv * a.n_sc > g.n_vh_max) { h->err = "internal: tc scratch too small"; return HERMES_ESTATE; }
  h->n_vh = g.Hkv * a.n_sc;
  {
    TcProf p(h, HERMES_K_SCORE_STATS, s);
    a.tpg = tpg1;
    k_tc_stats<<<n_cta1, kTcStatsThreads, kTcSmemBytes, s>>>(tmap_q, st->tmap_k, a);
  }
  {
    TcProf p(h, HERMES_K_SCORE_COLSUM, s);
    a.tpg = tpg2;
    k_tc_colsum<<<n_cta2, kTcColsumThreads, kTcSmemBytes, s>>>(tmap_q, st->tmap_k, a);
  }
  return HERMES_OK;
}

}  // namespace hk
