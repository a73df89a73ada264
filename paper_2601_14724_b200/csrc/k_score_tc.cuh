// a1 -- attention importance W (Eq. 2) on the 5th-gen tensor cores: bf16, head_dim 128.
//
// Same two-pass recompute as the CUDA-core path (k_score_simt.cuh), as ONE persistent, warp-specialised
// tcgen05 kernel (k_tc_score) fed by TMA, with fp32 accumulators in TMEM:
//   pass 1 (tc_pass1)  : D[row, tok] = Q_blk K_tile^T, probe rows on TMEM lanes -> each thread owns one
//                        probe row and keeps its running (max, sum exp2) over the tokens: no cross-lane work.
//   pass 2 (tc_pass2)  : D[tok, row] = K_tile Q^T, tokens on TMEM lanes -> each thread owns one token and
//                        accumulates sum_r exp2(s * scale - c_r), c_r = m_r + log2 Z_r merged from pass 1.
// A "group" = (stream, scored layer, KV head, row super-chunk of <= 512 probe rows); its Q rows stay in
// shared memory while the 128-token K tiles of the group stream through a TMA ring.  The flattened
// (group, tile) space is cut into equal contiguous ranges, one per CTA (<= #SM CTAs, 1 CTA/SM).
//
// Both passes are bound by the exp2 rate of the XU pipe (16 results / clk / SM), and every MUFU, TMEM
// load and mbarrier poll of an SM sub-partition shares one in-order MIO queue.  Hence the shape of the
// epilogue: 16 warps (4 per sub-partition), each working through 32-column blocks with the TMEM load of
// the NEXT block (and the barrier poll it may need) issued before the exp2 burst of the current one, and
// no integer division (I2F / MUFU.RCP would queue behind the exp2 traffic) anywhere in a loop.
#pragma once
#include "host_state.cuh"
#include "tc_ptx.cuh"

namespace hk {

constexpr int kTcRowsMax = 512;                 // probe rows resident per group (Q tile <= 128 KB)
constexpr int kTcTile = 128;                    // tokens per K tile (both passes)
constexpr int kTcKStage = kTcTile * 256;        // bytes per K tile: 128 tokens x 128 dims bf16
constexpr int kTcKStagesMax = 4;                // K ring depth: as many 32 KB stages as fit beside the Q rows
constexpr int kTcSmemMax = 232448;              // 227 KB dynamic shared memory per CTA
constexpr int kTcEpiWarps = 16;                 // epilogue warps: 4 per SM sub-partition / TMEM lane quarter
constexpr int kTcCtlWarps = 4;                  // warpgroup 0: producer, MMA issuer, V mover, (idle)
constexpr int kTcThreads = (kTcCtlWarps + kTcEpiWarps) * 32;   // the epilogue warps are warpgroups 1-4
constexpr int kTcRegsLaunch = 96;                // registers per thread at launch (640 threads)
constexpr int kTcRegsCtl = 64, kTcRegsEpi = 104; // setmaxnreg: warpgroup 0 releases registers, the epilogue warps take them
// setmaxnreg.inc draws only on registers released by setmaxnreg.dec in the same CTA -- it spins forever otherwise
static_assert((kTcRegsLaunch - kTcRegsCtl) * kTcCtlWarps >= (kTcRegsEpi - kTcRegsLaunch) * kTcEpiWarps, "register pool");
constexpr int kTcMoverRingMax = 32768;          // shared-memory staging of the V mover: at most 32 KB ...
constexpr int kTcMoverRowsMin = 8;              // ... and at least 8 rows per batch, else the move does not ride
constexpr int kTcSegTiles = 4;                  // pass 1: 128-token tiles per segment (one partial pair per
                                                // segment, so the merge order never depends on the CTA schedule)

struct TcArgs {
  Geom g;
  int cur, Tn, P;
  float scale_log2;
  int R, RS, n_sc;          // probe rows per KV head (G*P), rows per super-chunk, super-chunks per KV head
  int tpg;                  // 128-token tiles per group
  int n_groups;             // B * Ls * Hkv * n_sc
  int spg;                  // pass 1: 512-token segments per group = partial (m, z) slots per probe row
  int q_half_bytes;         // shared-memory bytes of one 64-column half of the group's Q rows (64-row boxes)
  int n_kst;                // K ring stages
  // deferred V compaction of the PREVIOUS update, moved by one warp per CTA while this update is scored
  const char* v_base;       // V cache base, or NULL: nothing pending
  const int32_t* v_kept;    // [B*L][budget] kept lists of the previous update
  int v_src_buf, v_row_bytes;
  int v_n_new;              // layer-dependent budgets: rows layer l held after the previous update = lay_T[l] - v_n_new
  int v_ring_bytes;         // staging ring of the mover: a whole number of rows (tc_ring_bytes)
  // layer-dependent budgets (k_tc_score<true>): every scored layer has its own tile / segment count; pre_s / pre_t are the
  // prefix sums of segments / tiles over the (stream, scored layer) blocks of Hkv * n_sc groups, [B * Ls + 1] each
  const int32_t* pre_s;
  const int32_t* pre_t;
  int U1, U2;               // schedule units of pass 1 (segments) and of pass 2 (tiles)
};

// ---- schedule: CTA c owns flattened units [c*U/nC, (c+1)*U/nC) -----------------------------------
__host__ __device__ inline int tc_unit_begin(int U, int n_cta, int c) { return int(((long long)U * c) / n_cta); }

// Group coordinates (super-chunk, KV head, scored layer, stream), advanced without integer division.
struct TcCursor {
  int sc, kvh, ls, bq;
  __device__ inline void init(const TcArgs& a, int gi) {
    const int Ls = a.g.L - a.g.n_shallow;
    sc = gi % a.n_sc;
    kvh = (gi / a.n_sc) % a.g.Hkv;
    const int bls = gi / (a.n_sc * a.g.Hkv);
    ls = bls % Ls; bq = bls / Ls;
  }
  __device__ inline void next(const TcArgs& a) {
    if (++sc == a.n_sc) { sc = 0; if (++kvh == a.g.Hkv) { kvh = 0; if (++ls == a.g.L - a.g.n_shallow) { ls = 0; ++bq; } } }
  }
  __device__ inline int bl(const TcArgs& a) const { return bq * a.g.L + a.g.n_shallow + ls; }
  __device__ inline int rs_valid(const TcArgs& a) const { return min(a.RS, a.R - sc * a.RS); }
  __device__ inline int stat_row0(const TcArgs& a) const { return kvh * a.R + sc * a.RS; }
};

// Tiles / segments of a group: the launch's, or (kLb) those of its layer's own candidate count T_l.
template <bool kLb> __device__ __forceinline__ int tc_tiles_of(const TcArgs& a, int T_l) { return kLb ? (T_l + kTcTile - 1) / kTcTile : a.tpg; }
template <bool kLb> __device__ __forceinline__ int tc_segs_of(const TcArgs& a, int T_l) {
  return kLb ? (tc_tiles_of<true>(a, T_l) + kTcSegTiles - 1) / kTcSegTiles : a.spg;
}
template <bool kLb> __device__ __forceinline__ int tc_layer_T(const TcArgs& a, const TcCursor& g) {
  return kLb ? layer_T(a.g, a.g.n_shallow + g.ls, a.Tn) : a.Tn;
}
// Schedule unit u -> (group, unit inside the group).  kSeg: units are pass-1 segments, else pass-2 tiles.
template <bool kLb, bool kSeg>
__device__ inline void tc_locate(const TcArgs& a, int u, int& gi, int& x) {
  if (!kLb) { const int upg = kSeg ? a.spg : a.tpg; gi = u / upg; x = u - gi * upg; return; }
  const int32_t* pre = kSeg ? a.pre_s : a.pre_t;
  int lo = 0, hi = a.g.B * (a.g.L - a.g.n_shallow);        // pre[lo] <= u < pre[hi] (u == total: the empty range at the end)
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(pre + mid) <= u) lo = mid; else hi = mid; }
  const int ngb = a.g.Hkv * a.n_sc, base = __ldg(pre + lo), upg = (__ldg(pre + lo + 1) - base) / ngb;
  const int gb = (u - base) / upg;
  gi = lo * ngb + gb; x = u - base - gb * upg;
}

struct TcSmem {
  uint8_t* q;        // [2 halves][q_half_bytes / 128 rows][128 B], 128B-swizzled
  uint8_t* k;        // K ring: [stage][2 halves][128 tokens][128 B]
  float* c;          // [512] per-row c_r (pass 2)
  float4* xch;       // [2][8][32] pass-1 exchange between the two token-half warps of a row block quarter
  uint8_t* ring;     // V mover staging (v_ring_bytes; only when a compaction is pending)
  float2* xch2;      // [2][2][32] pass-1 exchange between the even- / odd-tile lane quarters of a half-full row block
  uint64_t* bars;    // mbarriers
  uint32_t* tmem;    // TMEM base address written by tcgen05.alloc
};
__host__ __device__ inline int tc_smem_bytes(int q_half_bytes, int n_kst, int ring_bytes) {
  return ring_bytes + 1024 + 2 * q_half_bytes + n_kst * kTcKStage + kTcRowsMax * 4 + 8192 + 1024 + 256 + 16;
}
// Staging ring of the V mover: what is left beside the Q rows and a 2-stage K ring, in whole rows, <= 32 rows and <= 32 KB;
// 0 = fewer than kTcMoverRowsMin rows fit (the move then goes through k_gather).
__host__ __device__ inline int tc_ring_bytes(int q_half_bytes, int row_bytes) {
  const int avail = kTcSmemMax - tc_smem_bytes(q_half_bytes, 2, 0);
  int rows = avail / row_bytes;
  if (rows > 32) rows = 32;
  if (rows * row_bytes > kTcMoverRingMax) rows = kTcMoverRingMax / row_bytes;
  return rows >= kTcMoverRowsMin ? rows * row_bytes : 0;
}
__device__ inline TcSmem tc_carve(uint8_t* raw, const TcArgs& a) {
  uint8_t* p = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(raw) + 1023) & ~uintptr_t(1023));
  TcSmem s;
  s.q = p; p += 2 * a.q_half_bytes;
  s.k = p; p += a.n_kst * kTcKStage;
  s.ring = p; p += a.v_ring_bytes;
  s.c = reinterpret_cast<float*>(p); p += kTcRowsMax * 4;
  s.xch = reinterpret_cast<float4*>(p); p += 8192;
  s.xch2 = reinterpret_cast<float2*>(p); p += 1024;
  s.bars = reinterpret_cast<uint64_t*>(p); p += 256;
  s.tmem = reinterpret_cast<uint32_t*>(p);
  return s;
}

struct TcBars {
  uint64_t *k_full, *k_empty, *t_full, *t_empty, *q_full, *q_empty, *v_full;
};
__device__ inline TcBars tc_bars(const TcSmem& s) {
  TcBars b;
  b.k_full = s.bars; b.k_empty = s.bars + kTcKStagesMax;
  b.t_full = s.bars + 2 * kTcKStagesMax; b.t_empty = b.t_full + 2;
  b.q_full = b.t_empty + 2; b.q_empty = b.q_full + 1; b.v_full = b.q_empty + 1;
  return b;
}
__device__ inline uint32_t tc_prologue(const TcSmem& s, const TcBars& b, const TcArgs& a, const CUtensorMap* tq, const CUtensorMap* tk) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(tq); ptx::prefetch_tmap(tk);
    for (int i = 0; i < a.n_kst; ++i) { ptx::mbar_init(&b.k_full[i], 1); ptx::mbar_init(&b.k_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&b.t_full[i], 1); ptx::mbar_init(&b.t_empty[i], kTcEpiWarps); }
    ptx::mbar_init(b.q_full, 1); ptx::mbar_init(b.q_empty, 1); ptx::mbar_init(b.v_full, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc(s.tmem, 512);
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  return *s.tmem;
}

// Pipeline state a thread carries from pass 1 into pass 2 (ring slot / phase of the K ring, TMEM stage /
// phase, number of Q loads so far); which fields a thread uses depends on its role.
struct TcRole { int ks = 0, kph = 0, as = 0, aph = 0, n_q = 0; };

// TMA producer (one thread), identical for both passes: the 128-token K tiles of units [u0, u1) and the
// Q rows of each group the CTA touches (both 64-column halves, 64-row boxes).  kSeg: unit = (group,
// segment of kTcSegTiles tiles); otherwise unit = (group, tile).  A new group's first K tile is requested
// before the Q buffer is waited for, so it is in flight while the old group's MMAs drain.
template <bool kSeg, bool kLb>
__device__ inline void tc_producer(const TcSmem& s, const TcBars& b, const CUtensorMap* tq, const CUtensorMap* tk,
                                   const TcArgs& a, int u0, int u1, TcRole& st) {
  int ks = st.ks, kph = st.kph, n_q = st.n_q;
  bool new_group = true;
  int x, gi0;
  tc_locate<kLb, kSeg>(a, u0, gi0, x);
  TcCursor g; g.init(a, gi0);
  int T_l = tc_layer_T<kLb>(a, g);
  for (int u = u0; u < u1; ++u) {
    const int upg = kSeg ? tc_segs_of<kLb>(a, T_l) : tc_tiles_of<kLb>(a, T_l);
    const int t0 = kSeg ? x * kTcSegTiles : x, t1 = kSeg ? min(tc_tiles_of<kLb>(a, T_l), t0 + kTcSegTiles) : x + 1;
    const int bl = g.bl(a);
    for (int t = t0; t < t1; ++t) {
      ptx::mbar_wait(&b.k_empty[ks], kph ^ 1);
      ptx::mbar_expect_tx(&b.k_full[ks], kTcKStage);
      const int row = int((size_t(bl) * 2 + a.cur) * a.g.cap) + t * kTcTile;
      for (int h = 0; h < 2; ++h)
        for (int bx = 0; bx < 2; ++bx)
          ptx::tma_load_2d(s.k + ks * kTcKStage + h * 16384 + bx * 8192, tk, &b.k_full[ks], g.kvh * 128 + h * 64, row + bx * 64);
      if (++ks == a.n_kst) { ks = 0; kph ^= 1; }
      if (new_group) {
        if (n_q > 0) ptx::mbar_wait(b.q_empty, (n_q - 1) & 1);
        const int n_box = (g.rs_valid(a) + 63) >> 6;
        const int q_row0 = bl * a.g.Hq * a.P + g.stat_row0(a);
        ptx::mbar_expect_tx(b.q_full, uint32_t(n_box) * 2 * 8192);
        for (int h = 0; h < 2; ++h)
          for (int bx = 0; bx < n_box; ++bx)
            ptx::tma_load_2d(s.q + h * a.q_half_bytes + bx * 8192, tq, b.q_full, h * 64, q_row0 + bx * 64);
        ++n_q; new_group = false;
      }
    }
    if (++x == upg) { x = 0; g.next(a); new_group = true; if (kLb) T_l = tc_layer_T<true>(a, g); }
  }
  st.ks = ks; st.kph = kph; st.n_q = n_q;
}

// =====================================================================================================
// pass 1: per probe row, partial (max, sum exp2) over this CTA's token range of the group.
// D[row, tok] = Q_blk K_tile^T: probe rows on TMEM lanes, so every epilogue thread owns one probe row.
// A TMEM stage (256 columns) holds a "half-group" = 2 row blocks x 128 tokens; epilogue warp
// (row block rbl, 64-token half th, lane quarter lg) takes its 64 columns as two 32-column blocks.
// =====================================================================================================
template <bool kEpi, bool kLb>
__device__ __forceinline__ void tc_pass1(const TcSmem& s, const TcBars& b, const CUtensorMap* tmap_q, const CUtensorMap* tmap_k,
                                         const TcArgs& a, uint32_t tmem_base, TcRole& st) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int U = a.U1;                                                    // schedule unit = (group, segment)
  const int s0 = tc_unit_begin(U, gridDim.x, blockIdx.x), s1 = tc_unit_begin(U, gridDim.x, blockIdx.x + 1);

  if (!kEpi && warp == 0) {
    if (lane == 0) tc_producer<true, kLb>(s, b, tmap_q, tmap_k, a, s0, s1, st);
  } else if (!kEpi && warp == 1) {
    // ---------------- MMA issuer: the whole warp runs the loop, one elected lane issues ----------------
    const uint32_t idesc = ptx::idesc_bf16_f32(128, kTcTile);
    const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(s.q)), k_lo = ptx::smem_desc_lo(ptx::smem_u32(s.k));
    const uint32_t q_half16 = uint32_t(a.q_half_bytes) >> 4;
    int ks = st.ks, kph = st.kph, as = st.as, aph = st.aph, n_q = st.n_q;
    bool new_group = true;
    int x, gi0;
    tc_locate<kLb, true>(a, s0, gi0, x);
    TcCursor g; g.init(a, gi0);
    int T_l = tc_layer_T<kLb>(a, g);
    for (int u = s0; u < s1; ++u) {
      const int n_rb = (g.rs_valid(a) + 127) >> 7;
      const bool shift = g.rs_valid(a) > 384 && g.rs_valid(a) <= 448;
      if (new_group) { ptx::mbar_wait(b.q_full, n_q & 1); ++n_q; new_group = false; }
      const bool last_seg_of_group = (u + 1 == s1) || x + 1 == tc_segs_of<kLb>(a, T_l);
      const int t_end = min(tc_tiles_of<kLb>(a, T_l), (x + 1) * kTcSegTiles);
      for (int t = x * kTcSegTiles; t < t_end; ++t) {
        ptx::mbar_wait(&b.k_full[ks], kph);
        const uint32_t kb_lo = k_lo + uint32_t(ks) * (kTcKStage >> 4);
        for (int hg = 0; 2 * hg < n_rb; ++hg) {
          ptx::mbar_wait(&b.t_empty[as], aph ^ 1);
          ptx::tc_fence_after();
          const uint32_t qa_lo = q_lo + uint32_t(2 * hg) * 1024u, d0 = tmem_base + as * 256;
          const bool two = 2 * hg + 1 < n_rb;
          // a fourth row block that is at most half full alternates between the lower (even tiles) and the
          // upper (odd tiles) 64 TMEM lanes -- the A tile then starts 64 rows earlier -- so that all four SM
          // sub-partitions carry the same exp2 load (see the epilogue)
          const uint32_t sh = (shift && hg == 1 && (t & 1)) ? 512u : 0u;
          if (ptx::elect_one()) {
#pragma unroll
            for (int kk = 0; kk < 8; ++kk)
              ptx::mma_bf16_lohi(d0, qa_lo + (kk >> 2) * q_half16 + (kk & 3) * 2,
                                 kb_lo + (kk >> 2) * 1024u + (kk & 3) * 2, ptx::kSmemDescHiSw128, idesc, kk > 0);
            if (two) {
#pragma unroll
              for (int kk = 0; kk < 8; ++kk)
                ptx::mma_bf16_lohi(d0 + kTcTile, qa_lo + 1024u - sh + (kk >> 2) * q_half16 + (kk & 3) * 2,
                                   kb_lo + (kk >> 2) * 1024u + (kk & 3) * 2, ptx::kSmemDescHiSw128, idesc, kk > 0);
            }
            ptx::mma_commit(&b.t_full[as]);
          }
          __syncwarp();
          if (++as == 2) { as = 0; aph ^= 1; }
        }
        if (ptx::elect_one()) {
          ptx::mma_commit(&b.k_empty[ks]);
          if (last_seg_of_group && t + 1 == t_end) ptx::mma_commit(b.q_empty);
        }
        __syncwarp();
        if (++ks == a.n_kst) { ks = 0; kph ^= 1; }
      }
      if (++x == tc_segs_of<kLb>(a, T_l)) { x = 0; g.next(a); new_group = true; if (kLb) T_l = tc_layer_T<true>(a, g); }
    }
    st.ks = ks; st.kph = kph; st.as = as; st.aph = aph; st.n_q = n_q;
  } else if (kEpi) {
    // ---------------- epilogue: one probe row x 64 tokens per thread per stage ----------------
    const int e = warp - kTcCtlWarps, rbl = e >> 3, th = (e >> 2) & 1, lg = warp & 3;
    const uint32_t t_addr = tmem_base + (uint32_t(lg * 32) << 16) + rbl * kTcTile + th * 64;
    int as = st.as, aph = st.aph;
    float m0 = -INFINITY, z0 = 0.f, m1 = -INFINITY, z1 = 0.f;            // running (max, sum) per half-group
    float v[64];
    // online (max, sum exp2) update with this thread's 64 tokens of one stage
    auto fold = [&](int n_valid, float& m_run, float& z_run) {
      if (n_valid < 64) {                                                // ragged last tile of the group
#pragma unroll
        for (int j = 0; j < 64; ++j) if (j >= n_valid) v[j] = -INFINITY;
      }
      float mx[4] = {v[0], v[1], v[2], v[3]};
#pragma unroll
      for (int j = 4; j < 64; j += 4) {
        mx[0] = fmaxf(mx[0], v[j]); mx[1] = fmaxf(mx[1], v[j + 1]);
        mx[2] = fmaxf(mx[2], v[j + 2]); mx[3] = fmaxf(mx[3], v[j + 3]);
      }
      const float m_new = fmaxf(m_run, fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * a.scale_log2);
      float sm[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int j = 0; j < 64; ++j) v[j] = fmaf(v[j], a.scale_log2, -m_new);
#pragma unroll
      for (int j = 0; j < 64; ++j) v[j] = fast_exp2(v[j]);
#pragma unroll
      for (int j = 0; j < 64; j += 4) { sm[0] += v[j]; sm[1] += v[j + 1]; sm[2] += v[j + 2]; sm[3] += v[j + 3]; }
      z_run = z_run * fast_exp2(m_run - m_new) + ((sm[0] + sm[1]) + (sm[2] + sm[3]));
      m_run = m_new;
    };
    int x, gi, n_done = 0;
    tc_locate<kLb, true>(a, s0, gi, x);
    TcCursor g; g.init(a, gi);
    // candidates of the group's layer: a.Tn, or (kLb) this layer's own count under layer-dependent budgets (DESIGN f4), which
    // also sets its tile and segment counts.  A template flag, not a run-time test: one more live register in this loop
    // spills (+2 us at configs[1])
    int T_l = tc_layer_T<kLb>(a, g);
    // tell pass 2 (of this or a neighbouring CTA) that `n_done` more segments of group gi are in memory
    auto publish = [&]() {
      __threadfence();
      __syncwarp();
      if (lane == 0) atomicAdd(a.g.seg_cnt + gi, unsigned(n_done));
      n_done = 0;
    };
    for (int u = s0; u < s1; ++u) {
      const int rs_valid = g.rs_valid(a);
      const bool two = rs_valid > 256;                                   // the group has a second half-group
      const bool act0 = rbl * 128 + lg * 32 < rs_valid, act1 = (2 + rbl) * 128 + lg * 32 < rs_valid;
      // half-full fourth row block: lanes 0-63 hold it on even tiles, lanes 64-127 on odd tiles (see the MMA warp)
      const bool shift = rs_valid > 384 && rs_valid <= 448 && rbl == 1;
      const bool act1_odd = lg >= 2 && 384 + (lg - 2) * 32 < rs_valid;
      const int t_end = min(tc_tiles_of<kLb>(a, T_l), (x + 1) * kTcSegTiles);
      for (int t = x * kTcSegTiles; t < t_end; ++t) {
        const int n_valid = T_l - (t * kTcTile + th * 64);
#pragma unroll
        for (int hg = 0; hg < 2; ++hg) {
          if (hg == 1 && !two) break;
          const bool act = (hg == 0 ? act0 : (shift && (t & 1)) ? act1_odd : act1) && n_valid > 0;
          ptx::mbar_wait(&b.t_full[as], aph);
          ptx::tc_fence_after();
          if (act) {
            ptx::tmem_ld32(t_addr + as * 256, v);
            ptx::tmem_ld32(t_addr + as * 256 + 32, v + 32);
            ptx::tmem_ld_wait();
          }
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(&b.t_empty[as]);               // accumulators are in registers
          if (++as == 2) { as = 0; aph ^= 1; }
          if (act) { if (hg == 0) fold(n_valid, m0, z0); else fold(n_valid, m1, z1); }
        }
      }
      // segment done: the two token-half warps of a (row block, lane quarter) merge through shared memory
      // (double-buffered by segment parity, one 64-thread barrier), then one partial per (segment, row)
      {
        const int pair = rbl * 4 + lg;
        float4* xch = s.xch + ((u & 1) * 8 + pair) * 32 + lane;
        if (th == 1) *xch = make_float4(m0, z0, m1, z1);
        ptx::named_bar_sync(2 + pair, 64);
        if (th == 0) {
          const float4 o = *xch;
          const float ma = fmaxf(m0, o.x), mb = fmaxf(m1, o.z);            // this half always saw a token: finite
          // a row / half that saw no token is (-inf, 0): keep it that way instead of exp2(-inf + inf)
          const float za = ma == -INFINITY ? 0.f : z0 * fast_exp2(m0 - ma) + o.y * fast_exp2(o.x - ma);
          const float zb = mb == -INFINITY ? 0.f : z1 * fast_exp2(m1 - mb) + o.w * fast_exp2(o.z - mb);
          float2* part = reinterpret_cast<float2*>(a.g.partial) +
                         (size_t(g.bl(a)) * a.spg + x) * (a.g.Hq * a.g.p_max) + g.stat_row0(a);
          const int row_a = rbl * 128 + lg * 32 + lane, row_b = row_a + 256;
          if (row_a < rs_valid) part[row_a] = make_float2(ma, za);
          if (!shift) {
            if (row_b < rs_valid) part[row_b] = make_float2(mb, zb);
          } else {
            // the odd-tile share of rows 384 + (lg - 2) * 32 + lane sits in lane quarter lg >= 2: hand it to quarter lg - 2
            float2* x2 = s.xch2 + ((u & 1) * 2 + (lg & 1)) * 32 + lane;
            if (lg >= 2) *x2 = make_float2(mb, zb);
            ptx::named_bar_sync(10 + (lg & 1), 64);
            if (lg < 2 && row_b < rs_valid) {
              const float2 o = *x2;
              const float m = fmaxf(mb, o.x);                            // both -inf: a segment past this layer's candidates
              part[row_b] = make_float2(m, m == -INFINITY ? 0.f : zb * fast_exp2(mb - m) + o.y * fast_exp2(o.x - m));
            }
          }
        }
        m0 = m1 = -INFINITY; z0 = z1 = 0.f;
      }
      ++n_done;
      if (++x == tc_segs_of<kLb>(a, T_l)) { publish(); x = 0; ++gi; g.next(a); if (kLb) T_l = tc_layer_T<true>(a, g); }
    }
    if (n_done > 0) publish();
    st.as = as; st.aph = aph;
  }
}

// Pass-2 group prologue: merges each probe row's per-(segment, half) (m, z) partials of pass 1 in slot
// order into c_r = m_r + log2 Z_r (shared memory); rows past the group get +inf: exp2(-inf) = 0.
// 16 independent loads in flight per thread.  Kept out of line so its registers do not weigh on the hot loop.
__device__ __noinline__ void tc_merge_rows(const float2* pr, int n_slot, int rows_total, int rs_valid, float* c_out, int et,
                                           int row0, int P, int skip_below) {
  for (int i = et; i < kTcRowsMax; i += kTcEpiWarps * 32) {
    float c = INFINITY;
    // skip_below > 0 (deep layers, DESIGN f3): probe rows below it (row = query head * P + probe index) are left out
    if (i < rs_valid && (row0 + i) % P >= skip_below) {
      const float2* p2 = pr + i;
      float m = -INFINITY, zz = 0.f;
      for (int j0 = 0; j0 < n_slot; j0 += 16) {
        float2 pv[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) pv[j] = __ldcg(p2 + size_t(min(j0 + j, n_slot - 1)) * rows_total);   // always in range: no branch
#pragma unroll
        for (int j = 0; j < 16; ++j) if (j0 + j >= n_slot) pv[j] = make_float2(-INFINITY, 0.f);
        float mc = m;
#pragma unroll
        for (int j = 0; j < 16; ++j) mc = fmaxf(mc, pv[j].x);
        zz = m == -INFINITY ? 0.f : zz * fast_exp2(m - mc);
#pragma unroll
        for (int j = 0; j < 16; ++j) zz += pv[j].y * fast_exp2(pv[j].x - mc);
        m = mc;
      }
      c = m + log2f(zz);
    }
    c_out[i] = c;
  }
}

// =====================================================================================================
// pass 2: per token, sum over the group's probe rows of exp2(s * scale - c_r).
// D[tok, row] = K_tile Q^T: tokens on TMEM lanes, so every epilogue thread owns one token; a TMEM stage
// holds a chunk of <= 256 probe rows of the 128-token tile; epilogue warp (lane quarter lg, column
// quarter cq) takes 32-column blocks cq and cq + 4 of the chunk.
// =====================================================================================================
template <bool kEpi, bool kLb>
__device__ __forceinline__ void tc_pass2(const TcSmem& s, const TcBars& b, const CUtensorMap* tmap_q, const CUtensorMap* tmap_k,
                                         const TcArgs& a, uint32_t tmem_base, TcRole& st) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int U = a.U2;
  const int u0 = tc_unit_begin(U, gridDim.x, blockIdx.x), u1 = tc_unit_begin(U, gridDim.x, blockIdx.x + 1);

  if (!kEpi && warp == 0) {
    if (lane == 0) tc_producer<false, kLb>(s, b, tmap_q, tmap_k, a, u0, u1, st);
  } else if (!kEpi && warp == 1) {
    // ---------------- MMA issuer: the whole warp runs the loop, one elected lane issues ----------------
    const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(s.q)), k_lo = ptx::smem_desc_lo(ptx::smem_u32(s.k));
    const uint32_t q_half16 = uint32_t(a.q_half_bytes) >> 4;
    int ks = st.ks, kph = st.kph, as = st.as, aph = st.aph, n_q = st.n_q;
    bool new_group = true;
    int t, gi0;
    tc_locate<kLb, false>(a, u0, gi0, t);
    TcCursor g; g.init(a, gi0);
    int T_l = tc_layer_T<kLb>(a, g);
    for (int u = u0; u < u1; ++u) {
      const int rs32 = (g.rs_valid(a) + 31) & ~31;
      if (new_group) { ptx::mbar_wait(b.q_full, n_q & 1); ++n_q; new_group = false; }
      ptx::mbar_wait(&b.k_full[ks], kph);
      const uint32_t ka_lo = k_lo + uint32_t(ks) * (kTcKStage >> 4);
      for (int c0 = 0; c0 < rs32; c0 += 256) {                           // probe-row chunks of <= 256 columns
        const int nc = min(256, rs32 - c0);
        ptx::mbar_wait(&b.t_empty[as], aph ^ 1);
        ptx::tc_fence_after();
        const uint32_t idesc = ptx::idesc_bf16_f32(128, nc);
        const uint32_t qb_lo = q_lo + uint32_t(c0) * 8u;                 // c0 rows x 128 B >> 4
        if (ptx::elect_one()) {
#pragma unroll
          for (int kk = 0; kk < 8; ++kk)
            ptx::mma_bf16_lohi(tmem_base + as * 256, ka_lo + (kk >> 2) * 1024u + (kk & 3) * 2,
                               qb_lo + (kk >> 2) * q_half16 + (kk & 3) * 2, ptx::kSmemDescHiSw128, idesc, kk > 0);
          ptx::mma_commit(&b.t_full[as]);
        }
        __syncwarp();
        if (++as == 2) { as = 0; aph ^= 1; }
      }
      const bool last_of_group = (u + 1 == u1) || t + 1 == tc_tiles_of<kLb>(a, T_l);
      if (ptx::elect_one()) {
        ptx::mma_commit(&b.k_empty[ks]);
        if (last_of_group) ptx::mma_commit(b.q_empty);
      }
      __syncwarp();
      if (++ks == a.n_kst) { ks = 0; kph ^= 1; }
      if (++t == tc_tiles_of<kLb>(a, T_l)) { t = 0; g.next(a); new_group = true; if (kLb) T_l = tc_layer_T<true>(a, g); }
    }
  } else if (kEpi) {
    // ---------------- epilogue: one token per thread; warp (lane quarter lg, column quarter cq) ----------------
    const int e = warp - kTcCtlWarps, cq = e >> 2, lg = warp & 3;
    const int tok_in_tile = lg * 32 + lane;
    const uint32_t t_addr = tmem_base + (uint32_t(lg * 32) << 16) + cq * 32;
    int as = st.as, aph = st.aph;
    float v[32];
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    bool new_group = true;
    int t, gi, rs32 = 0, T_l = a.Tn;
    tc_locate<kLb, false>(a, u0, gi, t);
    float* col = nullptr;                                                // this warp's column-sum slot of the group
    TcCursor g; g.init(a, gi);
    // seg_cnt[group] counts 16 (epilogue warps) per finished pass-1 segment of THIS update (k_append zeroes the counters);
    // a group is complete at 16 x its segment count (layer-dependent budgets: its layer's own)
    // sum over the 32 probe rows [col0, col0 + 32) of this token (32 registers live: no spills in this loop --
    // a local-memory load would queue behind the exp2 traffic like every other MIO instruction)
    auto fold = [&](int col0) {
      const float4* c4 = reinterpret_cast<const float4*>(s.c + col0);
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
    for (int u = u0; u < u1; ++u) {
      if (new_group) {
        // all pass-1 segments of the group must be in memory (they come from this CTA and its schedule
        // neighbours, none of which ever waits during pass 1, and every CTA of the grid is resident)
        if (kLb) T_l = tc_layer_T<true>(a, g);
        if (lane == 0) {
          const unsigned seg_target = unsigned(tc_segs_of<kLb>(a, T_l)) * kTcEpiWarps;
          unsigned seen;
          do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(a.g.seg_cnt + gi) : "memory"); }
          while (seen < seg_target);
        }
        __syncwarp();
        ptx::named_bar_sync(1, kTcEpiWarps * 32);                        // everyone is done with the old c_r
        const int bl = g.bl(a), rows_total = a.g.Hq * a.g.p_max;
        tc_merge_rows(reinterpret_cast<const float2*>(a.g.partial) + size_t(bl) * a.spg * rows_total + g.stat_row0(a),
                      tc_segs_of<kLb>(a, T_l), rows_total, g.rs_valid(a), s.c, threadIdx.x - kTcCtlWarps * 32, g.sc * a.RS, a.P,
                      g.ls >= a.g.L - a.g.n_shallow - a.g.n_deep ? a.g.probe_deep_begin : 0);
        ptx::named_bar_sync(1, kTcEpiWarps * 32);
        rs32 = (g.rs_valid(a) + 31) & ~31;
        col = a.g.colsum + (size_t(bl) * a.g.n_vh_max + (g.kvh * a.n_sc + g.sc) * 4 + cq) * a.g.cap;
        new_group = false;
      }
      for (int c0 = 0; c0 < rs32; c0 += 256) {
        const int nc = min(256, rs32 - c0);
        const bool b0 = cq * 32 < nc, b1 = (cq + 4) * 32 < nc;           // this warp's 32-column blocks: cq and cq + 4
        ptx::mbar_wait(&b.t_full[as], aph);
        ptx::tc_fence_after();
        if (b0) {
          ptx::tmem_ld32(t_addr + as * 256, v);
          ptx::tmem_ld_wait();
          fold(c0 + cq * 32);
        }
        if (b1) {
          ptx::tmem_ld32(t_addr + as * 256 + 128, v);
          ptx::tmem_ld_wait();
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&b.t_empty[as]);                 // this warp's share of the stage is in registers
        if (++as == 2) { as = 0; aph ^= 1; }
        if (b1) fold(c0 + (cq + 4) * 32);
      }
      // per-(KV head, super-chunk, column quarter) column sum of this token; k_wsum adds the slots in order
      const int tok = t * kTcTile + tok_in_tile;
      if (tok < T_l) col[tok] = (acc[0] + acc[1]) + (acc[2] + acc[3]);
      acc[0] = acc[1] = acc[2] = acc[3] = 0.f;
      if (++t == tc_tiles_of<kLb>(a, T_l)) { t = 0; ++gi; g.next(a); new_group = true; }
    }
  }
}

// V mover (warp 2): compaction of V needs no arithmetic and nothing in the scoring of the NEXT update
// reads V, so k_gather leaves V behind and this warp moves the kept rows V[kept[s]] -> V'[s] of the previous update
// with 1D bulk copies (global -> shared -> global) while the tensor / XU pipes score: one row per lane, one
// mbarrier wait per batch.  The CTA's share is ~1200 rows of 1 KB over ~200 us: a few GB/s per SM.
__device__ inline void tc_v_mover(const TcSmem& s, const TcBars& b, const TcArgs& a) {
  const int lane = threadIdx.x & 31;
  const int budget = a.g.budget, rb = a.v_row_bytes;
  const int per = a.v_ring_bytes / rb;                                    // rows per batch (8..32)
  const long long n_rows = (long long)a.g.B * a.g.L * budget;
  const long long r0 = n_rows * blockIdx.x / gridDim.x, r1 = n_rows * (blockIdx.x + 1) / gridDim.x;
  int bl = int(r0 / budget), sl = int(r0 - (long long)bl * budget) + lane;   // this lane's (slab, slot); no division below
  int l = bl % a.g.L;
  int ph = 0;
  for (long long i0 = r0; i0 < r1; i0 += per) {
    while (sl >= budget) { sl -= budget; ++bl; if (++l == a.g.L) l = 0; }
    const bool on = lane < per && i0 + lane < r1;
    int src = -1;
    if (on) src = __ldcg(a.v_kept + size_t(bl) * budget + sl);            // < 0: summary-token slot, not a copy
    // layer-dependent budgets: `budget` is the list stride (the largest layer's); this layer holds fewer rows
    if (on && a.g.lay_T != nullptr && sl >= __ldg(a.g.lay_T + l) - a.v_n_new) src = -1;
    const unsigned m = __ballot_sync(0xffffffffu, on && src >= 0);
    if (m != 0) {
      if (lane == 0) ptx::mbar_expect_tx(b.v_full, uint32_t(__popc(m)) * rb);
      __syncwarp();
      uint8_t* slot = s.ring + lane * rb;
      if (on && src >= 0)
        ptx::bulk_load(slot, a.v_base + ((size_t(bl) * 2 + a.v_src_buf) * a.g.cap + src) * rb, rb, b.v_full);
      ptx::mbar_wait(b.v_full, ph); ph ^= 1;
      if (on && src >= 0) {
        ptx::bulk_store(const_cast<char*>(a.v_base) + ((size_t(bl) * 2 + (a.v_src_buf ^ 1)) * a.g.cap + sl) * rb, slot, rb);
        ptx::bulk_commit();
      }
      ptx::bulk_wait_read0();                                             // staging slots may be overwritten
      __syncwarp();
    }
    sl += per;
  }
  ptx::bulk_wait0();                                                      // every row is in global memory
}

// =====================================================================================================
// One persistent kernel runs both passes: every CTA works through its pass-1 range, then its pass-2
// range of the same flattened (group, token) space, keeping TMEM, barriers and the K ring alive.  Pass 2
// of a group only waits (on seg_cnt) for the pass-1 segments of that group, i.e. for this CTA and its
// schedule neighbours -- there is no grid-wide barrier.  Requires every CTA resident: the launch is cooperative
// (gridDim.x <= #SMs; the runtime refuses it on an SM-limited context, and the caller falls back to the CUDA-core path).
// =====================================================================================================
// kLb: layer-dependent budgets (per-layer candidate counts); the uniform-budget instantiation is the one bench.py times.
template <bool kLb>
__global__ void __launch_bounds__(kTcThreads, 1)
k_tc_score(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k, TcArgs a) {
  extern __shared__ uint8_t smem_raw[];
  const TcSmem s = tc_carve(smem_raw, a);
  const TcBars b = tc_bars(s);
  const uint32_t tmem_base = tc_prologue(s, b, a, &tmap_q, &tmap_k);
  pdl_wait();                       // the chunk's K rows come from k_append
  if (threadIdx.x == 0) pdl_launch_dependents();
  // 20 warps start with 96 registers each; warpgroup 0 hands 32 of them to the 16 epilogue warps (+8 each).  Each side stays in
  // its own branch until the end of the kernel (ptxas bounds registers per region between setmaxnreg and the join).
  TcRole st;
  if ((threadIdx.x >> 5) < kTcCtlWarps) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kTcRegsCtl));
    if ((threadIdx.x >> 5) == 2 && a.v_base != nullptr) tc_v_mover(s, b, a);
    tc_pass1<false, kLb>(s, b, &tmap_q, &tmap_k, a, tmem_base, st);
    tc_pass2<false, kLb>(s, b, &tmap_q, &tmap_k, a, tmem_base, st);
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kTcRegsEpi));
    tc_pass1<true, kLb>(s, b, &tmap_q, &tmap_k, a, tmem_base, st);
    tc_pass2<true, kLb>(s, b, &tmap_q, &tmap_k, a, tmem_base, st);
  }
  ptx::tc_fence_before();
  __syncthreads();
  if ((threadIdx.x >> 5) == 1) ptx::tmem_dealloc(tmem_base, 512);
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
  int occ = 0;
  if (cudaFuncSetAttribute(k_tc_score<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemMax) != cudaSuccess ||
      cudaFuncSetAttribute(k_tc_score<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemMax) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_tc_score<false>, kTcThreads, kTcSmemMax) != cudaSuccess || occ < 1) {
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

// Can a pending V compaction ride in the scoring launch of (Tn, P)?  The mover needs its staging ring beside a
// K ring of >= 2 stages, and it must finish before the scoring does: one warp per CTA moves ~32 rows per 3 us
// (one bulk-copy round trip), while the scoring runs at ~2.75e6 exp2 per us on the whole chip (both measured).
inline bool tc_v_ride_ok(const hermes_t* h, int Tn, int P) {
  const Geom& g = h->geom;
  const TcState* st = static_cast<const TcState*>(h->tc_state);
  const int R = g.G * P;
  int n_sc = (R + kTcRowsMax - 1) / kTcRowsMax;
  const int RS = ((R + n_sc - 1) / n_sc + 31) & ~31;
  const int q_half = (RS + 63) / 64 * 8192;
  const int ring = tc_ring_bytes(q_half, int(h->lay.row_bytes));
  if (ring == 0) return false;
  const double score_us = 2.0 * g.Hq * P * double(Tn) * (g.L - g.n_shallow) * g.B / 2.75e6;
  const double rows_per_cta = double(g.B) * g.L * g.budget / st->n_sm;
  const double per = double(ring / int(h->lay.row_bytes));
  return score_us >= 1.25 * (rows_per_cta / per * 3.0);
}

constexpr int kTcNotResident = 1;   // tc_score: the cooperative launch was refused; the caller scores on the CUDA-core path

struct TcProf {   // same event bracketing as hermes_api.cu's Prof, local to this header
  hermes_t* h; int id; cudaStream_t s;
  TcProf(hermes_t* h_, int id_, cudaStream_t s_) : h(h_), id(id_), s(s_) {
    if (h->profiling) { cudaEventRecord(h->timer.beg[id], s); h->timer.ran[id] = true; }
    ++h->last_launches;
  }
  ~TcProf() { if (h->profiling) cudaEventRecord(h->timer.end[id], s); }
};

inline int tc_score(hermes_t* h, const void* q_probe, int Tn, int n_new, int P, float scale_log2, cudaStream_t s, bool move_v) {
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
  a.tpg = (Tn + kTcTile - 1) / kTcTile;
  a.spg = (a.tpg + kTcSegTiles - 1) / kTcSegTiles;
  long long U1 = (long long)a.n_groups * a.spg, U2 = (long long)a.n_groups * a.tpg;
  if (U2 > INT_MAX / 2) { h->err = "tcgen05 scoring: too many (group, tile) units"; return HERMES_ECAPACITY; }
  if (h->lb) {
    // layer-dependent budgets: Tn is the largest scored layer's count (it sizes the partial-slot stride a.spg); every scored
    // layer runs its own ceil(T_l / 128) tiles, and the CTAs split the sums of those.  Prefix sums per (stream, scored layer)
    // block of Hkv * n_sc groups, uploaded stream-ordered (pageable source: staged when the call returns)
    const int Ls = g.L - g.n_shallow, nb = g.B * Ls, ngb = g.Hkv * a.n_sc;
    std::vector<int32_t> pre(2 * size_t(nb + 1), 0);
    for (int i = 0; i < nb; ++i) {
      const int T_l = h->lay_len[g.n_shallow + i % Ls] + n_new;
      const int tiles = (T_l + kTcTile - 1) / kTcTile, segs = (tiles + kTcSegTiles - 1) / kTcSegTiles;
      pre[i + 1] = pre[i] + ngb * segs;
      pre[nb + 1 + i + 1] = pre[nb + 1 + i] + ngb * tiles;
    }
    U1 = pre[nb]; U2 = pre[2 * nb + 1];
    int32_t* dev = reinterpret_cast<int32_t*>(h->ws + h->lay.tc_pre);
    if (cudaMemcpyAsync(dev, pre.data(), pre.size() * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) {
      h->err = "tcgen05 scoring: upload of the per-layer schedule failed"; return HERMES_ECUDA;
    }
    a.pre_s = dev; a.pre_t = dev + nb + 1;
  }
  a.U1 = int(U1); a.U2 = int(U2);
  // every CTA must be resident (pass 2 waits on pass-1 progress of other CTAs): at most one CTA per SM
  const int n_cta = int(std::min<long long>(st->n_sm, U1));
  if (a.spg > h->lay.n_part_max || g.Hkv * a.n_sc * 4 > g.n_vh_max || a.n_groups > g.B * g.L * g.n_vh_max) { h->err = "internal: tc scratch too small"; return HERMES_ESTATE; }
  h->n_vh = g.Hkv * a.n_sc * 4;
  a.q_half_bytes = (a.RS + 63) / 64 * 8192;
  // a pending V compaction of the previous update rides in this launch (tc_v_mover)
  a.v_base = move_v ? static_cast<const char*>(g.vc) : nullptr;
  a.v_kept = g.kept; a.v_src_buf = h->v_src_buf; a.v_row_bytes = int(h->lay.row_bytes); a.v_n_new = n_new;
  a.v_ring_bytes = move_v ? tc_ring_bytes(a.q_half_bytes, a.v_row_bytes) : 0;
  if (move_v && a.v_ring_bytes == 0) { h->err = "internal: V mover ring does not fit (tc_v_ride_ok)"; return HERMES_ESTATE; }
  a.n_kst = std::min(kTcKStagesMax, (kTcSmemMax - tc_smem_bytes(a.q_half_bytes, 0, a.v_ring_bytes)) / kTcKStage);
  if (a.n_kst < 2) { h->err = "tcgen05 scoring: shared memory too small for the K ring"; return HERMES_ESTATE; }
  const int smem = tc_smem_bytes(a.q_half_bytes, a.n_kst, a.v_ring_bytes);
  {
    TcProf p(h, HERMES_K_SCORE_STATS, s);
    // cooperative: pass 2 of a CTA waits for pass-1 statistics of other CTAs, so all of them must be resident
    const cudaError_t e = h->lb ? launch_pdl_coop(k_tc_score<true>, dim3(n_cta), dim3(kTcThreads), size_t(smem), s, tmap_q, st->tmap_k, a)
                                : launch_pdl_coop(k_tc_score<false>, dim3(n_cta), dim3(kTcThreads), size_t(smem), s, tmap_q, st->tmap_k, a);
    if (e == cudaErrorCooperativeLaunchTooLarge) {             // not every CTA can be resident (SM-limited context): no spin-waits then
      (void)cudaGetLastError();
      return kTcNotResident;
    }
    if (e != cudaSuccess) { h->err = std::string("tcgen05 scoring launch: ") + cudaGetErrorString(e); return HERMES_ECUDA; }
  }
  return HERMES_OK;
}

}  // namespace hk
