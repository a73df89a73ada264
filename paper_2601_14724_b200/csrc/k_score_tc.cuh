// a1 -- attention importance W (Eq. 2) on the 5th-gen tensor cores: bf16, head_dim 128.
//
// Same two-pass recompute as the CUDA-core path (k_score_simt.cuh), as ONE persistent, warp-specialised
// tcgen05 kernel (k_tc_score) fed by TMA, with fp32 accumulators in TMEM:
//   pass 1 (tc_pass1)  : D[row, tok] = Q_blk K_tile^T, probe rows on TMEM lanes -> each thread owns one
//                        probe row and keeps its running (max, sum exp2) over the tokens: no cross-lane work.
//   pass 2 (tc_pass2)  : D[tok, row] = K_tile Q^T, tokens on TMEM lanes -> each thread owns one token and
//                        accumulates sum_r exp2(s * scale - c_r), c_r = m_r + log2 Z_r merged from pass 1.
// A "group" = (stream, scored layer, KV head, row super-chunk of <= 512 probe rows); its Q rows stay in
// shared memory while the 128-token K tiles of the group stream through a TMA ring.
//
// Schedule: layer-major BATCHES.  The scored (stream, layer) slabs are cut into batches of a few slabs whose keys
// fit the L2 cache; every CTA takes an equal contiguous share of a batch's (group, token) units, and works through
//     pass 1 (batch 0), pass 1 (batch 1), pass 2 (batch 0), pass 1 (batch 2), pass 2 (batch 1), ...
// so that pass 2 re-reads a batch's keys from L2 instead of HBM, and pass 1 always runs one batch ahead of the
// pass 2 that needs its row statistics (a group's pass 2 waits only for that group's pass-1 segments, published
// through seg_cnt: there is no grid-wide barrier).  Requires gridDim.x <= #SMs with every CTA resident.
//
// Movers (tc_mover): gather-compaction (a5) and the delta rotary correction (a7) of the PREVIOUS update ride in
// this launch.  Nothing in this update reads V, and a slab's compacted K is only needed once the schedule reaches
// that slab, so two warps per CTA move the kept rows old buffer -> shared memory ring -> (K: rotate in place)
// -> current buffer with 1D bulk copies while the tensor / XU pipes score; the TMA producer waits on a per-slab
// row counter (kready) before it loads keys a mover still has to deliver.  HBM and the SMs are busy together.
//
// Both passes are bound by the exp2 rate of the XU pipe (16 results / clk / SM), and every MUFU, TMEM
// load and mbarrier poll of an SM sub-partition shares one in-order MIO queue.  Hence the shape of the
// epilogue: 16 warps (4 per sub-partition), no register spills, and no integer division (I2F / MUFU.RCP would
// queue behind the exp2 traffic) anywhere in a hot loop.
#pragma once
#include "host_state.cuh"
#include "k_gather.cuh"
#include "tc_ptx.cuh"

namespace hk {

constexpr int kTcRowsMax = 512;                 // probe rows resident per group (Q tile <= 128 KB)
constexpr int kTcTile = 128;                    // tokens per K tile (both passes)
constexpr int kTcKStage = kTcTile * 256;        // bytes per K tile: 128 tokens x 128 dims bf16
constexpr int kTcKStagesMax = 4;                // K ring depth: as many 32 KB stages as fit beside the Q rows
constexpr int kTcSmemMax = 232448;              // 227 KB dynamic shared memory per CTA
constexpr int kTcEpiWarps = 16;                 // epilogue warps: 4 per SM sub-partition / TMEM lane quarter
constexpr int kTcCtlWarps = 4;                  // warpgroup 0: producer, MMA issuer, two movers
constexpr int kTcThreads = (kTcCtlWarps + kTcEpiWarps) * 32;   // the epilogue warps are warpgroups 1-4
constexpr int kTcRegsLaunch = 96;                // registers per thread at launch (640 threads)
constexpr int kTcRegsCtl = 64, kTcRegsEpi = 104; // setmaxnreg: warpgroup 0 releases registers, the epilogue warps take them
// setmaxnreg.inc draws only on registers released by setmaxnreg.dec in the same CTA -- it spins forever otherwise
static_assert((kTcRegsLaunch - kTcRegsCtl) * kTcCtlWarps >= (kTcRegsEpi - kTcRegsLaunch) * kTcEpiWarps, "register pool");
constexpr int kTcSegTiles = 4;                  // pass 1: 128-token tiles per segment (one partial pair per
                                                // segment, so the merge order never depends on the CTA schedule)
constexpr int kMvSlotsMax = 12;                 // mover: ring slots (batches in flight) per mover warp
constexpr int kMvRowsMax = 8;                   // mover: rows per batch
constexpr int kMvLag = 2;                       // mover: store groups allowed in flight before their rows are published

struct TcArgs {
  Geom g;
  int cur, Tn, P;
  float scale_log2;
  int R, RS, n_sc;          // probe rows per KV head (G*P), rows per super-chunk, super-chunks per KV head
  int tpg;                  // 128-token tiles per group
  int spg;                  // pass 1: 512-token segments per group = partial (m, z) slots per probe row
  int gps;                  // groups per scored slab: Hkv * n_sc
  int n_slab;               // scored slabs: B * (L - n_shallow), in processing order (slab_of_order)
  int sb, ramp, n_batch;    // batches: `ramp` batches of 1, 2, 4, ... slabs, then batches of `sb` slabs
  int rot;                  // per-batch rotation of the CTA -> share map (spreads the remainders)
  int q_half_bytes;         // shared-memory bytes of one 64-column half of the group's Q rows (64-row boxes)
  int n_kst;                // K ring stages
  // deferred compaction of the PREVIOUS update, moved by two warps per CTA while this update is scored
  const char* mv_k;         // K cache base, or NULL: no K rows pending
  const char* mv_v;         // V cache base, or NULL: no V rows pending
  int mv_src_buf;           // buffer the kept rows still sit in (they go to mv_src_buf ^ 1 = the current one)
  int mv_k_ord0;            // K rows of the slabs with processing order >= mv_k_ord0 are pending
  int mv_rows, mv_slots;    // rows per batch, ring slots per mover warp
  int row_bytes;
};

// ---- schedule -----------------------------------------------------------------------------------
__host__ __device__ inline int tc_batch_slab(int ramp, int sb, int n_slab, int b) {   // first slab of batch b
  const int s = b <= ramp ? (1 << b) - 1 : (1 << ramp) - 1 + (b - ramp) * sb;
  return s < n_slab ? s : n_slab;
}
// Units [u0, u1) of batch b owned by this CTA; a unit is (group, segment) in pass 1 (upg = spg) and (group, tile)
// in pass 2 (upg = tpg), numbered globally as group * upg + index.
__device__ inline void tc_range(const TcArgs& a, int b, int upg, int& u0, int& u1) {
  const int s0 = tc_batch_slab(a.ramp, a.sb, a.n_slab, b), s1 = tc_batch_slab(a.ramp, a.sb, a.n_slab, b + 1);
  const long long U = (long long)(s1 - s0) * a.gps * upg;
  const int cc = int((blockIdx.x + (long long)b * a.rot) % gridDim.x);
  const int base = s0 * a.gps * upg;
  u0 = base + int(U * cc / gridDim.x);
  u1 = base + int(U * (cc + 1) / gridDim.x);
}

// Every role walks the same sequence of 2 n_batch items: pass 1 (0), pass 1 (1), pass 2 (0), pass 1 (2), pass 2 (1), ...,
// pass 2 (n - 1): pass 1 of batch b >= 1 is item 2b - 1, pass 2 of batch b <= n - 2 is item 2b + 2.
__device__ __forceinline__ bool tc_item_is_p1(int item, int n_batch) { return item == 0 || ((item & 1) && item != 2 * n_batch - 1); }
__device__ __forceinline__ int tc_item_batch(int item, int n_batch) {
  return item == 0 ? 0 : item == 2 * n_batch - 1 ? n_batch - 1 : (item & 1) ? (item + 1) >> 1 : (item >> 1) - 1;
}

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
  __device__ inline int order(const TcArgs& a) const { return bq * (a.g.L - a.g.n_shallow) + ls; }   // see slab_of_order
  __device__ inline int rs_valid(const TcArgs& a) const { return min(a.RS, a.R - sc * a.RS); }
  __device__ inline int stat_row0(const TcArgs& a) const { return kvh * a.R + sc * a.RS; }
};

struct TcSmem {
  uint8_t* q;        // [2 halves][q_half_bytes / 128 rows][128 B], 128B-swizzled
  uint8_t* k;        // K ring: [stage][2 halves][128 tokens][128 B]
  uint8_t* ring;     // movers: [2 warps][mv_slots][mv_rows][row_bytes] (only when a compaction is pending)
  float* c;          // [512] per-row c_r (pass 2)
  float4* xch;       // [2][8][32] pass-1 exchange between the two token-half warps of a row block quarter
  float2* xch2;      // [2][2][32] pass-1 exchange between the even- / odd-tile lane quarters of a half-full row block
  int4* mv_info;     // movers: [2 warps][mv_slots][mv_rows][2] what sits in each ring row
  uint64_t* bars;    // mbarriers
  int* wst;          // [2][32] per-warp state parked in shared memory: next schedule item, pass-1 segments folded
  uint32_t* tmem;    // TMEM base address written by tcgen05.alloc
};
constexpr int kMvInfoBytes = 32;                // per ring row: (source row, slot, slab, is-K) + the position deltas
// ring_rows: rows of the movers' staging ring (both warps), each `row_bytes` + kMvInfoBytes
__host__ __device__ inline int tc_smem_bytes(int q_half_bytes, int n_kst, int ring_rows, int row_bytes) {
  return 1024 + 2 * q_half_bytes + n_kst * kTcKStage + ring_rows * (row_bytes + kMvInfoBytes) + kTcRowsMax * 4 + 8192 + 1024 + 512 + 256 + 16;
}
__device__ inline TcSmem tc_carve(uint8_t* raw, const TcArgs& a) {
  uint8_t* p = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(raw) + 1023) & ~uintptr_t(1023));
  const int ring_rows = (a.mv_k || a.mv_v) ? 2 * a.mv_slots * a.mv_rows : 0;
  TcSmem s;
  s.q = p; p += 2 * a.q_half_bytes;
  s.k = p; p += a.n_kst * kTcKStage;
  s.ring = p; p += ring_rows * a.row_bytes;
  s.c = reinterpret_cast<float*>(p); p += kTcRowsMax * 4;
  s.xch = reinterpret_cast<float4*>(p); p += 8192;
  s.xch2 = reinterpret_cast<float2*>(p); p += 1024;
  s.mv_info = reinterpret_cast<int4*>(p); p += ring_rows * kMvInfoBytes;
  s.bars = reinterpret_cast<uint64_t*>(p); p += 512;
  s.wst = reinterpret_cast<int*>(p); p += 256;
  s.tmem = reinterpret_cast<uint32_t*>(p);
  return s;
}

struct TcBars {
  uint64_t *k_full, *k_empty, *t_full, *t_empty, *q_full, *q_empty, *mv_full;
};
__device__ inline TcBars tc_bars(const TcSmem& s) {
  TcBars b;
  b.k_full = s.bars; b.k_empty = s.bars + kTcKStagesMax;
  b.t_full = s.bars + 2 * kTcKStagesMax; b.t_empty = b.t_full + 2;
  b.q_full = b.t_empty + 2; b.q_empty = b.q_full + 1; b.mv_full = b.q_empty + 1;   // mv_full: [2][kMvSlotsMax]
  return b;
}
static_assert((2 * kTcKStagesMax + 4 + 2 + 2 * kMvSlotsMax) * 8 <= 512, "mbarrier space");

__device__ inline uint32_t tc_prologue(const TcSmem& s, const TcBars& b, const TcArgs& a, const CUtensorMap* tq, const CUtensorMap* tk) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(tq); ptx::prefetch_tmap(tk);
    for (int i = 0; i < a.n_kst; ++i) { ptx::mbar_init(&b.k_full[i], 1); ptx::mbar_init(&b.k_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&b.t_full[i], 1); ptx::mbar_init(&b.t_empty[i], kTcEpiWarps); }
    ptx::mbar_init(b.q_full, 1); ptx::mbar_init(b.q_empty, 1);
    for (int i = 0; i < 2 * kMvSlotsMax; ++i) ptx::mbar_init(&b.mv_full[i], 1);
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc(s.tmem, 512);
  if (threadIdx.x < 64) s.wst[threadIdx.x] = 0;
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  return *s.tmem;
}

// Pipeline state a thread carries from launch to exit (ring slot / phase of the K ring, TMEM stage / phase, number of
// Q loads so far, segments folded, last slab whose keys are known to be in place); which fields a thread uses
// depends on its role.
struct TcRole { int ks = 0, kph = 0, as = 0, aph = 0, n_q = 0, ready_ord = -1; };

// TMA producer (one thread), identical for both passes: the 128-token K tiles of units [u0, u1) and the
// Q rows of each group the CTA touches (both 64-column halves, 64-row boxes).  kSeg: unit = (group,
// segment of kTcSegTiles tiles); otherwise unit = (group, tile).  A new group's first K tile is requested
// before the Q buffer is waited for, so it is in flight while the old group's MMAs drain.
template <bool kSeg>
__device__ inline void tc_producer(const TcSmem& s, const TcBars& b, const CUtensorMap* tq, const CUtensorMap* tk,
                                   const TcArgs& a, int u0, int u1, TcRole& st) {
  if (u0 >= u1) return;
  const int upg = kSeg ? a.spg : a.tpg;
  int ks = st.ks, kph = st.kph, n_q = st.n_q;
  bool new_group = true;
  int x = u0 % upg;
  TcCursor g; g.init(a, u0 / upg);
  for (int u = u0; u < u1; ++u) {
    const int t0 = kSeg ? x * kTcSegTiles : x, t1 = kSeg ? min(a.tpg, t0 + kTcSegTiles) : x + 1;
    const int bl = g.bl(a);
    if (a.mv_k != nullptr && new_group) {
      // keys of this slab that a mover of this launch still has to deliver (every CTA's movers work through the
      // slabs in schedule order and never wait on anything but their own copies)
      const int ord = g.order(a);
      if (ord >= a.mv_k_ord0 && ord != st.ready_ord) {
        unsigned seen;
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(a.g.kready + bl) : "memory"); }
        while (seen < unsigned(a.g.budget));
        asm volatile("fence.proxy.async;" ::: "memory");        // the rows were written through the async proxy; so are the loads below
        st.ready_ord = ord;
      }
    }
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
    if (++x == upg) { x = 0; g.next(a); new_group = true; }
  }
  st.ks = ks; st.kph = kph; st.n_q = n_q;
}

// =====================================================================================================
// pass 1: per probe row, partial (max, sum exp2) over this CTA's token range of the group.
// D[row, tok] = Q_blk K_tile^T: probe rows on TMEM lanes, so every epilogue thread owns one probe row.
// A TMEM stage (256 columns) holds a "half-group" = 2 row blocks x 128 tokens; epilogue warp
// (row block rbl, 64-token half th, lane quarter lg) takes its 64 columns as two 32-column blocks.
// =====================================================================================================
template <bool kEpi>
__device__ __forceinline__ void tc_pass1(const TcSmem& s, const TcBars& b, const CUtensorMap* tmap_q, const CUtensorMap* tmap_k,
                                         const TcArgs& a, uint32_t tmem_base, TcRole& st, int batch, int tid) {
  const int warp = tid >> 5, lane = tid & 31;
  int s0, s1;                                                            // schedule unit = (group, segment)
  tc_range(a, batch, a.spg, s0, s1);

  if (!kEpi && warp == 0) {
    if (lane == 0) tc_producer<true>(s, b, tmap_q, tmap_k, a, s0, s1, st);
  } else if (!kEpi && warp == 1) {
    // ---------------- MMA issuer: the whole warp runs the loop, one elected lane issues ----------------
    if (s0 >= s1) return;
    const uint32_t idesc = ptx::idesc_bf16_f32(128, kTcTile);
    const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(s.q)), k_lo = ptx::smem_desc_lo(ptx::smem_u32(s.k));
    const uint32_t q_half16 = uint32_t(a.q_half_bytes) >> 4;
    int ks = st.ks, kph = st.kph, as = st.as, aph = st.aph, n_q = st.n_q;
    bool new_group = true;
    int x = s0 % a.spg;
    TcCursor g; g.init(a, s0 / a.spg);
    for (int u = s0; u < s1; ++u) {
      const int n_rb = (g.rs_valid(a) + 127) >> 7;
      const bool shift = g.rs_valid(a) > 384 && g.rs_valid(a) <= 448;
      if (new_group) { ptx::mbar_wait(b.q_full, n_q & 1); ++n_q; new_group = false; }
      const bool last_seg_of_group = (u + 1 == s1) || x + 1 == a.spg;
      const int t_end = min(a.tpg, (x + 1) * kTcSegTiles);
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
      if (++x == a.spg) { x = 0; g.next(a); new_group = true; }
    }
    st.ks = ks; st.kph = kph; st.as = as; st.aph = aph; st.n_q = n_q;
  } else if (kEpi) {
    // ---------------- epilogue: one probe row x 64 tokens per thread per stage ----------------
    if (s0 >= s1) return;
    const int e = warp - kTcCtlWarps, rbl = e >> 3, th = (e >> 2) & 1, lg = warp & 3;
    const uint32_t t_addr = tmem_base + (uint32_t(lg * 32) << 16) + rbl * kTcTile + th * 64;
    int as = st.as, aph = st.aph;
    float m0 = -INFINITY, z0 = 0.f, m1 = -INFINITY, z1 = 0.f;            // running (max, sum) per half-group
    float v[64];
    // online (max, sum exp2) update with this thread's 64 tokens of one stage
    auto fold = [&](int n_valid, float& m_run, float& z_run) __attribute__((always_inline)) {
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
    int x = s0 % a.spg, gi = s0 / a.spg, n_done = 0;
    TcCursor g; g.init(a, gi);
    // tell pass 2 (of this or a neighbouring CTA) that `n_done` more segments of group gi are in memory
    auto publish = [&]() __attribute__((always_inline)) {
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
      const int t_end = min(a.tpg, (x + 1) * kTcSegTiles);
      for (int t = x * kTcSegTiles; t < t_end; ++t) {
        const int n_valid = a.Tn - (t * kTcTile + th * 64);
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
        const int n_seg = s.wst[32 + warp];                                // segments folded so far (parked in shared memory:
        __syncwarp();                                                      // the loops above have no register to spare)
        if (lane == 0) s.wst[32 + warp] = n_seg + 1;
        float4* xch = s.xch + ((n_seg & 1) * 8 + pair) * 32 + lane;
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
            float2* x2 = s.xch2 + ((n_seg & 1) * 2 + (lg & 1)) * 32 + lane;
            if (lg >= 2) *x2 = make_float2(mb, zb);
            ptx::named_bar_sync(10 + (lg & 1), 64);
            if (lg < 2 && row_b < rs_valid) {
              const float2 o = *x2;
              const float m = fmaxf(mb, o.x);                            // a segment holds at least one tile: not both -inf
              part[row_b] = make_float2(m, zb * fast_exp2(mb - m) + o.y * fast_exp2(o.x - m));
            }
          }
        }
        m0 = m1 = -INFINITY; z0 = z1 = 0.f;
      }
      ++n_done;
      if (++x == a.spg) { publish(); x = 0; ++gi; g.next(a); }
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
template <bool kEpi>
__device__ __forceinline__ void tc_pass2(const TcSmem& s, const TcBars& b, const CUtensorMap* tmap_q, const CUtensorMap* tmap_k,
                                         const TcArgs& a, uint32_t tmem_base, TcRole& st, int batch, int tid) {
  const int warp = tid >> 5, lane = tid & 31;
  int u0, u1;
  tc_range(a, batch, a.tpg, u0, u1);

  if (!kEpi && warp == 0) {
    if (lane == 0) tc_producer<false>(s, b, tmap_q, tmap_k, a, u0, u1, st);
  } else if (!kEpi && warp == 1) {
    // ---------------- MMA issuer: the whole warp runs the loop, one elected lane issues ----------------
    if (u0 >= u1) return;
    const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(s.q)), k_lo = ptx::smem_desc_lo(ptx::smem_u32(s.k));
    const uint32_t q_half16 = uint32_t(a.q_half_bytes) >> 4;
    int ks = st.ks, kph = st.kph, as = st.as, aph = st.aph, n_q = st.n_q;
    bool new_group = true;
    int t = u0 % a.tpg;
    TcCursor g; g.init(a, u0 / a.tpg);
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
      const bool last_of_group = (u + 1 == u1) || t + 1 == a.tpg;
      if (ptx::elect_one()) {
        ptx::mma_commit(&b.k_empty[ks]);
        if (last_of_group) ptx::mma_commit(b.q_empty);
      }
      __syncwarp();
      if (++ks == a.n_kst) { ks = 0; kph ^= 1; }
      if (++t == a.tpg) { t = 0; g.next(a); new_group = true; }
    }
    st.ks = ks; st.kph = kph; st.as = as; st.aph = aph; st.n_q = n_q;
  } else if (kEpi) {
    // ---------------- epilogue: one token per thread; warp (lane quarter lg, column quarter cq) ----------------
    if (u0 >= u1) return;
    const int e = warp - kTcCtlWarps, cq = e >> 2, lg = warp & 3;
    const int tok_in_tile = lg * 32 + lane;
    const uint32_t t_addr = tmem_base + (uint32_t(lg * 32) << 16) + cq * 32;
    int as = st.as, aph = st.aph;
    float v[32];
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    bool new_group = true;
    int t = u0 % a.tpg, rs32 = 0, gi = u0 / a.tpg;
    float* col = nullptr;                                                // this warp's column-sum slot of the group
    TcCursor g; g.init(a, gi);
    const unsigned seg_target = unsigned(a.spg) * kTcEpiWarps;
    // sum over the 32 probe rows [col0, col0 + 32) of this token (32 registers live: no spills in this loop --
    // a local-memory load would queue behind the exp2 traffic like every other MIO instruction)
    auto fold = [&](int col0) __attribute__((always_inline)) {
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
        if (lane == 0) {
          unsigned seen;
          do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(a.g.seg_cnt + gi) : "memory"); }
          while (seen < seg_target);
        }
        __syncwarp();
        ptx::named_bar_sync(1, kTcEpiWarps * 32);                        // everyone is done with the old c_r
        const int bl = g.bl(a), rows_total = a.g.Hq * a.g.p_max;
        tc_merge_rows(reinterpret_cast<const float2*>(a.g.partial) + size_t(bl) * a.spg * rows_total + g.stat_row0(a),
                      a.spg, rows_total, g.rs_valid(a), s.c, tid - kTcCtlWarps * 32, g.sc * a.RS, a.P,
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
      if (tok < a.Tn) col[tok] = (acc[0] + acc[1]) + (acc[2] + acc[3]);
      acc[0] = acc[1] = acc[2] = acc[3] = 0.f;
      if (++t == a.tpg) { t = 0; ++gi; g.next(a); new_group = true; }
    }
    st.as = as; st.aph = aph;
  }
}

// =====================================================================================================
// Movers (warps 2 and 3): gather-compaction of the PREVIOUS update, K'[s] = rot(K[kept[s]], delta[s]) and
// V'[s] = V[kept[s]] (a5 + a7), from buffer mv_src_buf into the current one.  Every CTA owns the same slot range
// [M c / nC, M (c+1) / nC) of every slab (halved between its two mover warps), and works through the slabs in
// schedule order -- first K of all pending slabs, then V -- so that a slab's keys are complete early, when every
// CTA is done with its few rows of it.  Per warp a ring of mv_slots batches x mv_rows rows: 1D bulk copies
// global -> shared (one row per lane, one mbarrier per batch), rotation in place for K rows with a non-zero delta
// (same table, same fp32 no-FMA arithmetic and rounding as k_gather), bulk copy shared -> global.  Loads run
// mv_slots - kMvLag batches ahead of the batch being processed; a K row is published in kready[slab] once its
// store group has completed (kMvLag batches later), which is what the TMA producers wait for.
// =====================================================================================================
__device__ __forceinline__ void mv_rotate_row(const TcArgs& a, uint8_t* row, int d0, int d1, int d2, int lane,
                                              int& c_delta, float2 (&cs)[8]) {
  const Geom& g = a.g;
  const int jg = lane & 7, j0 = jg * 8;
  const bool unit_ok = g.n_axes == 1 || (((g.sec_t | g.sec_h) & 7) == 0);      // an 8-pair unit never straddles two M-RoPE sections
  const int dl = g.n_axes == 1 ? d0 : (j0 < g.sec_t ? d0 : (j0 < g.sec_t + g.sec_h ? d1 : d2));
  const int r = -dl;
  const bool fast = unit_ok && r > 0 && r < g.table_rows;
  if (fast && dl != c_delta) {
    const float4* tab = reinterpret_cast<const float4*>(g.rope_tab + size_t(r) * 64 + j0);
#pragma unroll
    for (int p = 0; p < 4; ++p) { const float4 t4 = __ldg(tab + p); cs[2 * p] = make_float2(t4.x, t4.y); cs[2 * p + 1] = make_float2(t4.z, t4.w); }
    c_delta = dl;
  }
  const int upr = g.Hkv * 8;
  for (int u = lane; u < upr; u += 32) {
    uint4* plo = reinterpret_cast<uint4*>(row + ((u >> 3) * 128 + j0) * 2);
    uint4* phi = plo + 8;
    uint4 lo = *plo, hi = *phi;
    if (fast) {
      float x[8], y[8];
      Elem<__nv_bfloat16>::unpack(lo, x);
      Elem<__nv_bfloat16>::unpack(hi, y);
#pragma unroll
      for (int p = 0; p < 8; ++p) rot_pair(x[p], y[p], cs[p].x, cs[p].y);
      lo = Elem<__nv_bfloat16>::pack(x);
      hi = Elem<__nv_bfloat16>::pack(y);
    } else if (unit_ok && dl == 0) {
      continue;                                                                  // this unit's axis did not move: bit-exact copy
    } else if (g.n_axes == 1) {
      const int dd[1] = {d0};
      rotate_unit<__nv_bfloat16, 1>(g, dd, j0, lo, hi);
    } else {
      const int dd[3] = {d0, d1, d2};
      rotate_unit<__nv_bfloat16, 3>(g, dd, j0, lo, hi);
    }
    *plo = lo; *phi = hi;
  }
}

__device__ __forceinline__ void tc_mover(const TcSmem& s, const TcBars& b, const TcArgs& a, int w) {
  const int lane = threadIdx.x & 31;
  const int R = a.mv_rows, S = a.mv_slots, rb = a.row_bytes, M = a.g.budget;
  uint8_t* ring = s.ring + size_t(w) * S * R * rb;
  uint64_t* full = b.mv_full + w * kMvSlotsMax;
  int4* info = s.mv_info + w * (S * R * 2);
  const int c0 = int((long long)M * blockIdx.x / gridDim.x), c1 = int((long long)M * (blockIdx.x + 1) / gridDim.x);
  const int mid = (c0 + c1 + 1) >> 1;
  const int sl0 = w == 0 ? c0 : mid, sl1 = w == 0 ? mid : c1, nper = sl1 - sl0;
  const int n_ord = a.g.B * a.g.L;
  const int nk = a.mv_k ? n_ord - a.mv_k_ord0 : 0, nv = a.mv_v ? n_ord : 0, nq = nk + nv;   // virtual slab sequence: K slabs, then V slabs
  if (nper <= 0 || nq <= 0) return;
  const int n_batch = int(((long long)nq * nper + R - 1) / R);
  const size_t slab_rows = size_t(a.g.cap);

  // this lane's next row to fetch indices for: (virtual slab q, slot); advanced by R rows per batch, no division
  int q = lane / nper, slot = sl0 + lane % nper, q_bl = -1, q_cached = -1;
  // indices of the batch about to be issued (prefetched one batch ahead of the issue)
  int n_src = -2, n_slot = 0, n_bl = 0, n_isk = 0, n_d0 = 0, n_d1 = 0, n_d2 = 0;
  auto fetch = [&]() __attribute__((always_inline)) {
    n_src = -2;                                                          // -2: no row (past the end / lane >= R)
    if (lane < R && q < nq) {
      if (q != q_cached) { q_bl = __ldg(a.g.ord2bl + (q < nk ? a.mv_k_ord0 + q : q - nk)); q_cached = q; }
      n_bl = q_bl; n_slot = slot; n_isk = q < nk;
      n_src = __ldcg(a.g.kept + size_t(q_bl) * M + slot);               // -1: summary-token slot, written by k_summary
      n_d0 = n_d1 = n_d2 = 0;
      if (n_isk) {
        const int32_t* dp = a.g.delta + size_t(q_bl) * a.g.n_axes * M + slot;
        n_d0 = __ldcg(dp);
        if (a.g.n_axes == 3) { n_d1 = __ldcg(dp + M); n_d2 = __ldcg(dp + 2 * M); }
      }
    }
    slot += R;
    while (slot >= sl1) { slot -= nper; ++q; }
  };
  unsigned loaded = 0u, phase = 0u;                                      // per ring slot: has loads in flight / mbarrier parity
  int is = 0;                                                            // ring slot of the next batch to issue
  auto issue = [&]() __attribute__((always_inline)) {
    const bool has = n_src >= 0;
    const unsigned m = __ballot_sync(0xffffffffu, has);
    if (lane < R) {
      info[(is * R + lane) * 2] = make_int4(n_src, n_slot, n_bl, n_isk);
      info[(is * R + lane) * 2 + 1] = make_int4(n_d0, n_d1, n_d2, 0);
    }
    if (m != 0u) {
      if (lane == 0) ptx::mbar_expect_tx(&full[is], uint32_t(__popc(m)) * rb);
      __syncwarp();
      if (has)
        ptx::bulk_load(ring + size_t(is * R + lane) * rb,
                       (n_isk ? a.mv_k : a.mv_v) + ((size_t(n_bl) * 2 + a.mv_src_buf) * slab_rows + n_src) * rb, rb, &full[is]);
      loaded |= 1u << is;
    } else {
      loaded &= ~(1u << is);
    }
    if (++is == S) is = 0;
  };

  fetch();
  const int ahead = S - kMvLag;                                          // batches issued before the first one is processed
  for (int j = 0; j < ahead && j < n_batch; ++j) { issue(); fetch(); }
  int ps = 0;                                                            // ring slot of the batch being processed
  int pub1 = -1, pub2 = -1;                                              // slabs of this lane's K rows stored 1 / 2 batches ago
  int c_delta = 0x7fffffff;
  float2 cs[8];
  auto publish = [&](int bl) __attribute__((always_inline)) {
    if (bl >= 0) {
      asm volatile("fence.proxy.async;" ::: "memory");
      __threadfence();
      atomicAdd(a.g.kready + bl, 1u);
    }
  };
  for (int bt = 0; bt < n_batch; ++bt) {
    if ((loaded >> ps) & 1u) { ptx::mbar_wait(&full[ps], (phase >> ps) & 1u); phase ^= 1u << ps; }
    __syncwarp();
    for (int r = 0; r < R; ++r) {                                        // rotate the K rows in place
      const int4 i0 = info[(ps * R + r) * 2];
      if (i0.x < 0 || i0.w == 0) continue;
      const int4 i1 = info[(ps * R + r) * 2 + 1];
      if ((i1.x | i1.y | i1.z) == 0) continue;                           // delta 0 on every axis: bit-exact copy
      mv_rotate_row(a, ring + size_t(ps * R + r) * rb, i1.x, i1.y, i1.z, lane, c_delta, cs);
    }
    ptx::fence_proxy_async();                                            // generic-proxy writes -> bulk-copy reads
    __syncwarp();
    int mine = -1;
    if (lane < R) {
      const int4 i0 = info[(ps * R + lane) * 2];
      if (i0.x >= 0)
        ptx::bulk_store(const_cast<char*>(i0.w ? a.mv_k : a.mv_v) + ((size_t(i0.z) * 2 + (a.mv_src_buf ^ 1)) * slab_rows + i0.y) * rb,
                        ring + size_t(ps * R + lane) * rb, rb);
      if (i0.x >= -1 && i0.w) mine = i0.z;                               // a K row (or the summary slot): counts towards kready
    }
    ptx::bulk_commit();
    if (++ps == S) ps = 0;
    // at most kMvLag store groups stay in flight: the ring slot of batch bt - kMvLag is free again, and its rows are in memory
    asm volatile("cp.async.bulk.wait_group %0;" ::"n"(kMvLag) : "memory");
    publish(pub2);
    pub2 = pub1; pub1 = mine;
    __syncwarp();
    if (bt + ahead < n_batch) { issue(); fetch(); }
  }
  ptx::bulk_wait0();                                                      // every row is in global memory
  publish(pub2); publish(pub1);
}
static_assert(kMvLag == 2, "tc_mover keeps exactly two batches of publish history");

// =====================================================================================================
// One persistent kernel runs both passes over all batches (see the schedule at the top), keeping TMEM, the barriers
// and the K ring alive throughout.  Requires gridDim.x <= #SMs (all CTAs resident).
// =====================================================================================================
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
  const int warp = threadIdx.x >> 5;
  if (warp < kTcCtlWarps) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kTcRegsCtl));
    if (warp >= 2) {
#ifndef HERMES_NO_MOVER
      if (a.mv_k != nullptr || a.mv_v != nullptr) tc_mover(s, b, a, warp - 2);
#endif
    } else {
#pragma unroll 1
      for (int item = 0; item < 2 * a.n_batch; ++item) {
        if (tc_item_is_p1(item, a.n_batch)) tc_pass1<false>(s, b, &tmap_q, &tmap_k, a, tmem_base, st, tc_item_batch(item, a.n_batch), int(threadIdx.x));
        else tc_pass2<false>(s, b, &tmap_q, &tmap_k, a, tmem_base, st, tc_item_batch(item, a.n_batch), int(threadIdx.x));
      }
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kTcRegsEpi));
    // the epilogue loops have no register to spare: the item counter is parked in shared memory while a pass runs
    for (;;) {
      const int item = *reinterpret_cast<volatile int*>(s.wst + warp);
      if (item >= 2 * a.n_batch) break;
      if (tc_item_is_p1(item, a.n_batch)) tc_pass1<true>(s, b, &tmap_q, &tmap_k, a, tmem_base, st, tc_item_batch(item, a.n_batch), int(threadIdx.x));
      else tc_pass2<true>(s, b, &tmap_q, &tmap_k, a, tmem_base, st, tc_item_batch(item, a.n_batch), int(threadIdx.x));
      __syncwarp();
      if ((threadIdx.x & 31) == 0) { volatile int* pi = s.wst + warp; *pi = *pi + 1; }
      __syncwarp();
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
  int diag_sb = 0, diag_know = -1;   // -DHERMES_DIAG builds only: HERMES_TC_SB / HERMES_TC_KNOW override the schedule
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
  st->n_sm = h->n_sm;
#ifdef HERMES_DIAG
  if (const char* e = getenv("HERMES_TC_SB")) st->diag_sb = atoi(e);
  if (const char* e = getenv("HERMES_TC_KNOW")) st->diag_know = atoi(e);
#endif
  const Geom& g = h->geom;
  if (!tc_make_map(st, &st->tmap_k, g.kc, uint64_t(g.row_elems), uint64_t(g.B) * g.L * 2 * g.cap)) {
    h->err = "cuTensorMapEncodeTiled(K cache) failed"; delete st; return false;
  }
  int occ = 0;
  if (cudaFuncSetAttribute(k_tc_score, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemMax) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_tc_score, kTcThreads, kTcSmemMax) != cudaSuccess || occ < 1) {
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

// Row super-chunks of the G*P probe rows that share a KV head.
inline void tc_row_split(const Geom& g, int P, int& R, int& RS, int& n_sc) {
  R = g.G * P;
  n_sc = (R + kTcRowsMax - 1) / kTcRowsMax;
  RS = ((R + n_sc - 1) / n_sc + 31) & ~31;            // rows per super-chunk, multiple of 32
  n_sc = (R + RS - 1) / RS;
}

// Mover ring geometry that fits beside the Q rows and a 2-stage K ring: rows per batch and slots per mover warp.
// Returns false if the ring would be too small to keep enough copies in flight.
inline bool tc_mover_ring(const hermes_t* h, int P, int& rows, int& slots) {
  const Geom& g = h->geom;
  int R, RS, n_sc;
  tc_row_split(g, P, R, RS, n_sc);
  const int q_half = (RS + 63) / 64 * 8192;
  const int rb = int(h->lay.row_bytes);
  const int avail = kTcSmemMax - tc_smem_bytes(q_half, 2, 0, rb);
  const int per_warp = avail / 2 / (rb + kMvInfoBytes);                  // rows per mover warp
  if (per_warp < 12) return false;
  rows = std::min(kMvRowsMax, std::max(1, per_warp / 6));
  slots = std::min(kMvSlotsMax, per_warp / rows);
  return slots >= 4;
}

// Can a pending compaction ride in the scoring launch of (Tn, P)?  The movers need their staging ring beside a
// K ring of >= 2 stages, and they must finish before the scoring does: a CTA's two mover warps sustain roughly
// 12 rows per us, while the scoring runs at ~2.75e6 exp2 per us on the whole chip (both measured).
inline bool tc_ride_ok(const hermes_t* h, int Tn, int P) {
  const Geom& g = h->geom;
  const TcState* st = static_cast<const TcState*>(h->tc_state);
  int rows, slots;
  if (!tc_mover_ring(h, P, rows, slots)) return false;
  const double score_us = 2.0 * g.Hq * P * double(Tn) * (g.L - g.n_shallow) * g.B / 2.75e6;
  const double rows_per_cta = double(g.B) * g.L * g.budget / st->n_sm;   // V rows (K rows ride only if there is room: tc_k_now)
  return score_us >= 1.25 * rows_per_cta / 12.0;
}

// How many slabs (in processing order) compact their K right away in k_gather instead of leaving it to the movers of the
// next scoring launch: the first slab of the schedule is needed at once, and the movers must deliver both K and V
// within the scoring time.
inline int tc_k_now(const hermes_t* h, int Tn, int P) {
  const Geom& g = h->geom;
  const TcState* st = static_cast<const TcState*>(h->tc_state);
  const int n_ord = g.B * g.L;
  if (st->diag_know >= 0) return std::min(st->diag_know, n_ord);
  if (!h->cfg.defer_k) return n_ord;
  const double score_us = 2.0 * g.Hq * P * double(Tn) * (g.L - g.n_shallow) * g.B / 2.75e6;
  const double rows_per_cta_slab = double(g.budget) / st->n_sm;
  // rows the movers can carry in 80 % of the launch, minus all of V
  const double k_slabs = (0.8 * score_us * 12.0) / rows_per_cta_slab - n_ord;
  const int deferred = int(std::max(0.0, std::min<double>(k_slabs, n_ord - 1)));
  return n_ord - deferred;
}

struct TcProf {   // same event bracketing as hermes_api.cu's Prof, local to this header
  hermes_t* h; int id; cudaStream_t s;
  TcProf(hermes_t* h_, int id_, cudaStream_t s_) : h(h_), id(id_), s(s_) {
    if (h->profiling) { cudaEventRecord(h->timer.beg[id], s); h->timer.ran[id] = true; }
    ++h->last_launches;
  }
  ~TcProf() { if (h->profiling) cudaEventRecord(h->timer.end[id], s); }
};

// move_v / move_k: the pending V rows / the pending K rows (slabs of order >= h->k_pending_ord0) ride in this launch.
inline int tc_score(hermes_t* h, const void* q_probe, int Tn, int P, float scale_log2, cudaStream_t s, bool move_v, bool move_k) {
  TcState* st = static_cast<TcState*>(h->tc_state);
  const Geom& g = h->geom;
  CUtensorMap tmap_q;
  if (!tc_make_map(st, &tmap_q, q_probe, 128, uint64_t(g.B) * g.L * g.Hq * P)) {
    h->err = "cuTensorMapEncodeTiled(Q_probe) failed (pointer must be 16-byte aligned)";
    return HERMES_EINVAL;
  }
  TcArgs a{};
  a.g = g; a.cur = h->cur; a.Tn = Tn; a.P = P; a.scale_log2 = scale_log2;
  tc_row_split(g, P, a.R, a.RS, a.n_sc);
  a.gps = g.Hkv * a.n_sc;
  a.n_slab = g.B * (g.L - g.n_shallow);
  a.tpg = (Tn + kTcTile - 1) / kTcTile;
  a.spg = (a.tpg + kTcSegTiles - 1) / kTcSegTiles;
  const long long n_groups = (long long)a.n_slab * a.gps;
  const long long U1 = n_groups * a.spg, U2 = n_groups * a.tpg;
  if (U2 > INT_MAX / 2) { h->err = "tcgen05 scoring: too many (group, tile) units"; return HERMES_ECAPACITY; }
  // every CTA must be resident (pass 2 waits on pass-1 progress of other CTAs): at most one CTA per SM
  const int n_cta = int(std::min<long long>(st->n_sm, U1));
  if (a.spg > h->lay.n_part_max || a.gps * 4 > g.n_vh_max) { h->err = "internal: tc scratch too small"; return HERMES_ESTATE; }
  h->n_vh = a.gps * 4;
  a.q_half_bytes = (a.RS + 63) / 64 * 8192;
  // batches: as many slabs as keep two batches of keys (pass 1 runs one batch ahead of pass 2) within ~1/2 of the L2,
  // but never fewer units than a few per CTA
  {
    const double slab_mb = double(Tn) * h->lay.row_bytes / 1e6;
    int sb = std::max(1, int(28.0 / slab_mb));
    const int min_sb = int((3LL * n_cta + (long long)a.gps * a.spg - 1) / ((long long)a.gps * a.spg));
    sb = std::max(sb, min_sb);
    if (st->diag_sb > 0) sb = st->diag_sb;
    sb = std::min(sb, a.n_slab);
    a.sb = sb;
    a.ramp = 0;
    if (move_k) while ((2 << a.ramp) <= sb && (1 << (a.ramp + 1)) - 1 < a.n_slab) ++a.ramp;   // 1, 2, 4, ... slabs first: keys arrive slab by slab
    const int first = std::min((1 << a.ramp) - 1, a.n_slab);
    a.n_batch = a.ramp + (a.n_slab - first + sb - 1) / sb;
    if (first >= a.n_slab) { a.n_batch = 0; while (tc_batch_slab(a.ramp, a.sb, a.n_slab, a.n_batch) < a.n_slab) ++a.n_batch; }
    a.rot = std::max(1, int(n_cta * 0.382));
  }
  a.mv_k = move_k ? static_cast<const char*>(g.kc) : nullptr;
  a.mv_v = move_v ? static_cast<const char*>(g.vc) : nullptr;
  a.mv_src_buf = h->pend_src_buf; a.mv_k_ord0 = h->k_pending_ord0; a.row_bytes = int(h->lay.row_bytes);
  int ring_rows = 0;
  if (move_k || move_v) {
    if (!tc_mover_ring(h, P, a.mv_rows, a.mv_slots)) { h->err = "internal: no room for the mover ring"; return HERMES_ESTATE; }
    ring_rows = 2 * a.mv_slots * a.mv_rows;
  }
  a.n_kst = std::min(kTcKStagesMax, (kTcSmemMax - tc_smem_bytes(a.q_half_bytes, 0, ring_rows, a.row_bytes)) / kTcKStage);
  if (a.n_kst < 2) { h->err = "tcgen05 scoring: shared memory too small for the K ring"; return HERMES_ESTATE; }
  const int smem = tc_smem_bytes(a.q_half_bytes, a.n_kst, ring_rows, a.row_bytes);
  {
    TcProf p(h, HERMES_K_SCORE_STATS, s);
    const cudaError_t e = launch_pdl(k_tc_score, dim3(n_cta), dim3(kTcThreads), size_t(smem), s, tmap_q, st->tmap_k, a);
    if (e != cudaSuccess) { h->err = std::string("tcgen05 scoring launch: ") + cudaGetErrorString(e); return HERMES_ECUDA; }
  }
  return HERMES_OK;
}

}  // namespace hk
