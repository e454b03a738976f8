// li_attn.cu -- li_sparse_attn for sm_100a: block-sparse flash attention over C_i = K^curr U S_i
// (Eq. 11), K/V tiles fetched IN PLACE from the frame-paged cache by TMA with the page
// as a tensor coordinate (replaces the paper's KV-Prep / Untile-Scatter copies).
//
// One CTA per SM = one query block (BLK query rows, padded to the 128-row UMMA tile) of one (call, head).
// What bounds this kernel on B200 is, in this order: shared-memory bandwidth (128 B/clk/SM), the MUFU (16 ex2/clk/SM)
// and the tensor pipe, all three within 1.5x of each other for d = 128.  Hence:
//   * Q lives in TENSOR MEMORY (written once through registers with tcgen05.st) and is the A operand of S = Q K^T,
//     so the tensor core never re-reads Q from shared memory; shared memory only sees each K/V byte twice
//     (TMA write + one MMA read).
//   * Every attended KV block is processed as two HALF-tiles of HALF = BLK/2 keys; S is TRIPLE-buffered in TMEM, the
//     tensor core runs up to three half-tiles ahead of the softmax warps, which therefore never wait for it:
//         QK(0) QK(1) QK(2) | PV(0) QK(3) | PV(1) QK(4) | ...   (K/V half-tiles are TMA-loaded in exactly this order
//                                                                into an 8-slot shared-memory ring)
//   * HALF/16 threads per query row (16 S columns each): the softmax is latency-bound, more warps hide it.
//   warps 0..4*NPART-1 : softmax + lazy correction + epilogue; warp w owns TMEM lanes 32(w%4).. and column part w/4
//   next warp          : TMA producer (one elected lane)
//   last warp          : TMEM allocation and the single-thread tcgen05.mma issuer
// TMEM (512 columns): [0,D/2) Q (bf16 pairs), [64,..) [128,..) [192,..) S buffers (fp32; P in bf16 overlays the first
// HALF/2 columns of its S buffer once S has been read), [256,256+D) O.
#include "li_internal.h"
#include "li_ptx.cuh"

namespace li {

#ifdef LI_TRACE
// debug timeline: CTA (0,0,0) records (event, half-tile, SM clock) per role into p.trace
#define TR(role, ev, t) do { if (p.trace != nullptr && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && lane == 0) { \
  int k_ = tr_n++; if (k_ < 1000) { long long c_; asm volatile("mov.u64 %0, %%clock64;" : "=l"(c_)); \
  p.trace[((role) * 1000 + k_) * 3 + 0] = (ev); p.trace[((role) * 1000 + k_) * 3 + 1] = (t); p.trace[((role) * 1000 + k_) * 3 + 2] = c_; } } } while (0)
#else
#define TR(role, ev, t) do { } while (0)
#endif

constexpr int kSelCap = 1024;       // selected-block indices staged in shared memory (rest read from global)
constexpr int kPageCap = 512;       // frame-list entries staged in shared memory (rest read from global)
constexpr int kTmemCols = 512;
// TMEM columns: Q | S of group 0, 1 | P of group 0, 1 | O of group 0, 1
constexpr int kQCol = 0, kSCol = 64, kSStride = 64, kPCol = 192, kPStride = 32, kOCol = 256, kOStride = 128;
constexpr int kStages = 4;          // slots of the K ring and of the V ring (half-tiles)
constexpr float kRescaleThreshold = 8.0f;   // log2 units: P stays <= 2^8 between lazy rescales
#ifndef LI_EMU_OF_4
#define LI_EMU_OF_4 0
#endif
#ifndef LI_EARLY_PREFETCH
#define LI_EARLY_PREFETCH 0
#endif
constexpr bool kEarlyPrefetch = LI_EARLY_PREFETCH != 0;   // prefetch the first half of S(t+2) in the middle of exp(t)
#ifndef LI_STAGGER
#define LI_STAGGER 800
#endif
constexpr long long kStaggerCycles = LI_STAGGER;          // start offset of softmax group 1 (SM clocks)
constexpr int kEmuOf4 = LI_EMU_OF_4;        // of every 4 column pairs, how many use the FMA-pipe exp2

template <int D, int BLK>
struct AttnCfg {
  static constexpr int HALF = BLK / 2;
  static constexpr int kSoftmaxWarps = 8;              // two groups of 4 warps (even / odd half-tiles)
  static constexpr int kProducerK = kSoftmaxWarps, kProducerV = kSoftmaxWarps + 1, kMmaWarp = kSoftmaxWarps + 2;   // + g
  static constexpr int kThreads = (kSoftmaxWarps + 4) * 32;
  static constexpr int kKVChunk = HALF * 128;          // bytes of one 64-column chunk of a K or V half-tile
  static constexpr int kStage = (D / 64) * kKVChunk;
  static constexpr int kOffRing = 0;
  static constexpr int kOffSel = 2 * kStages * kStage;               // K ring, then V ring
  static constexpr int kOffPages = kOffSel + kSelCap * 4;            // this call's frame list (page ids), staged once
  static constexpr int kOffXch = kOffPages + kPageCap * 4;           // (m, l) exchange between the groups: [2][2][128] floats
  static constexpr int kOffBar = kOffXch + 4 * 128 * 4;
  static constexpr int kTotal = kOffBar + 512 + 1024;                // + barriers + slack for 1024-B alignment
};

enum {
  BAR_FULL = 0,                        // +ring*kStages + slot   (ring 0 = K, 1 = V)
  BAR_EMPTY = BAR_FULL + 2 * kStages,  // +ring*kStages + slot
  BAR_S_FULL = BAR_EMPTY + 2 * kStages,  // +group: S(t) of the group is in tensor memory
  BAR_S_FREE = BAR_S_FULL + 2,         // +group: the group's softmax warps have S(t) in registers (4 arrivals)
  BAR_P_FULL = BAR_S_FREE + 2,         // +group: P(t) is in tensor memory (4 arrivals)
  BAR_PV_DONE = BAR_P_FULL + 2,        // +group: O[g] += P(t) V(t) has completed
  BAR_Q_READY = BAR_PV_DONE + 2,       // Q is in tensor memory (8 arrivals)
  BAR_O_FULL,                          // +group: the group's last PV has completed
  BAR_O_FULL1,
  BAR_COUNT
};

template <int D, int BLK>
__global__ void __launch_bounds__(AttnCfg<D, BLK>::kThreads, 1)
li_sparse_attn_kernel(const AttnParams p, const BatchMeta meta, const __grid_constant__ CUtensorMap tm_k_full,
                      const __grid_constant__ CUtensorMap tm_k_8, const __grid_constant__ CUtensorMap tm_v_full,
                      const __grid_constant__ CUtensorMap tm_v_8) {
  using L = AttnCfg<D, BLK>;
  constexpr int HALF = L::HALF;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *smem = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t sRing = smem_base + L::kOffRing;
  int32_t *sSel = reinterpret_cast<int32_t *>(smem + L::kOffSel);
  int32_t *sPages = reinterpret_cast<int32_t *>(smem + L::kOffPages);
  volatile float *sXch = reinterpret_cast<volatile float *>(smem + L::kOffXch);
  const uint32_t bar0 = smem_base + L::kOffBar;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + L::kOffBar + 8 * BAR_COUNT);
  auto bar = [&](int i) { return bar0 + 8u * i; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  int tr_n = 0; (void)tr_n;

  // ---- per-tile integer bookkeeping (Eq. 11 context assembly) ----
  const int foff = meta.frame_off[b];
  const int n_frames = meta.frame_off[b + 1] - foff;
  const int n_hist = n_frames - p.n_cur;
  const int L_hist = n_hist * p.T_f;
  const int L_cur = p.n_cur * p.T_f;
  const int M = (L_hist + BLK - 1) / BLK;
  const int Nc = (L_cur + BLK - 1) / BLK;
  const int64_t row_id = ((int64_t)b * p.H + h) * p.Nqb + i;
  const int valid_q = min(BLK, p.Lq - i * BLK);
  const int tail_cur = L_cur - (Nc - 1) * BLK, tail_hist = L_hist - (M - 1) * BLK;

  // ---- one-time setup (independent of the previous kernel: overlaps its tail under PDL) ----
  if (warp == L::kProducerK && lane == 0) {
    tma_prefetch_desc(&tm_k_full);
    tma_prefetch_desc(&tm_v_full);
    tma_prefetch_desc(&tm_k_8);
    tma_prefetch_desc(&tm_v_8);
    for (int k = 0; k < BAR_COUNT; ++k) {
      const bool by_group = k >= BAR_S_FREE && k < BAR_P_FULL + 2;       // S_FREE[2], P_FULL[2]: one arrival per warp
      mbar_init(bar(k), by_group ? 4 : (k == BAR_Q_READY ? L::kSoftmaxWarps : 1));
    }
    mbar_fence_init();
    fence_proxy_async();
  }
  if (warp == L::kMmaWarp) {
    tmem_alloc(smem_u32(tmem_slot), kTmemCols);
    tmem_relinquish();
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");     // sel_idx / sel_cnt come from li_block_select (PDL)
  const int cnt = p.sel_cnt[row_id];
  const int32_t *sel_row = p.sel_idx + row_id * p.kmax;
  const int n_tiles = Nc + cnt;
  for (int t = threadIdx.x; t < cnt && t < kSelCap; t += blockDim.x) sSel[t] = sel_row[t];
  // the frame list is read by the TMA producer for every half-tile: a global load there (L2 latency) would pace the
  // whole pipeline, so it is staged in shared memory once
  for (int t = threadIdx.x; t < n_frames && t < kPageCap; t += blockDim.x) sPages[t] = p.frame_idx[foff + t];
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  auto sel_at = [&](int jj) -> int { return jj < kSelCap ? sSel[jj] : sel_row[jj]; };
  auto page_at = [&](int f) -> int { return f < kPageCap ? sPages[f] : p.frame_idx[foff + f]; };
  // valid key columns of attended tile j (chunk blocks first, then the selected historical blocks).  Only two tiles
  // can be partial: the last chunk block, and the history tail block M-1, which (indices ascending) can only be the
  // last selected one -- so no per-tile lookup is needed.
  const int j_tail_hist = (cnt > 0 && sel_at(cnt - 1) == M - 1) ? n_tiles - 1 : -1;
  auto tile_valid = [&](int j) -> int {
    return j == Nc - 1 ? tail_cur : (j == j_tail_hist ? tail_hist : BLK);
  };
  // number of half-tiles with at least one valid key (a half-tile without any is skipped by every role)
  int T = 2 * n_tiles;
  if (Nc > 0 && tail_cur <= HALF) --T;
  if (j_tail_hist >= 0 && tail_hist <= HALF) --T;

  if (T > 0) {
    if (warp == L::kProducerK || warp == L::kProducerV) {
      // =============================== TMA producers ===============================
      // One warp streams the K half-tiles, one the V half-tiles, each into its own 4-slot ring in consumption
      // order.  The warp stays converged (index arithmetic on warp-uniform values); an elected lane issues the TMA.
      const int ring = warp == L::kProducerK ? 0 : 1;
      const CUtensorMap *tm_full = ring == 0 ? &tm_k_full : &tm_v_full;
      const CUtensorMap *tm_8 = ring == 0 ? &tm_k_8 : &tm_v_8;
      int j = 0, hh = 0;
      for (int t = 0; t < T; ++t) {
        // half-tile t = rows [t0, t0+HALF) of a region (history or chunk)
        const bool is_cur = j < Nc;
        const int blk = is_cur ? j : sel_at(j - Nc);
        const int f0 = is_cur ? n_hist : 0;            // first frame of the region inside this call's frame list
        const int region_len = is_cur ? L_cur : L_hist;
        const int t0 = blk * BLK + hh * HALF;
        if (hh == 0 && tile_valid(j) > HALF) hh = 1;
        else { ++j; hh = 0; }
        const int slot = t & (kStages - 1);
        const uint32_t dst = sRing + (ring * kStages + slot) * L::kStage, mb = bar(BAR_FULL + ring * kStages + slot);
        const int t_last = min(t0 + HALF, region_len) - 1;
        const int pg0 = t0 / p.T_f;
        const bool one_page = p.has_box_full && pg0 == t_last / p.T_f;
        const int page0 = page_at(f0 + pg0);
        mbar_wait(bar(BAR_EMPTY + ring * kStages + slot), ((t / kStages) & 1) ^ 1);
        TR(17 + ring, 1, t);
        if (elect_one()) {
          mbar_arrive_expect_tx(mb, HALF * D * 2);
          if (one_page) {
            // inside one page: one box per 64-column chunk; rows past the page end are zero-filled by the
            // hardware (a region always ends on a page boundary)
            const int row = t0 - pg0 * p.T_f;
#pragma unroll
            for (int c = 0; c < D / 64; ++c) tma_load_4d(dst + c * L::kKVChunk, tm_full, mb, c * 64, row, h, page0);
          } else {
            // straddles frames: 8-row pieces (one SWIZZLE_128B atom each, destinations stay 1024-B aligned)
            int cur_pg = pg0, page = page0;
            for (int g = 0; g < HALF / 8; ++g) {
              const int tt = t0 + g * 8;
              int row = p.T_f;             // out of bounds -> zeros
              if (tt < region_len) {
                const int pg = tt / p.T_f;
                if (pg != cur_pg) { cur_pg = pg; page = page_at(f0 + pg); }
                row = tt - pg * p.T_f;
              }
#pragma unroll
              for (int c = 0; c < D / 64; ++c)
                tma_load_4d(dst + c * L::kKVChunk + g * 1024, tm_8, mb, c * 64, row, h, page);
            }
          }
        }
        __syncwarp();
      }
    } else if (warp >= L::kMmaWarp) {
      // =============================== MMA issuers (one warp per softmax group) ===============================
      // Warp g issues, for its group's half-tiles t = g, g+2, ...:   QK(g) | QK(t+2) PV(t) | QK(t+4) PV(t+2) | ...
      // i.e. the next S is requested as soon as the softmax warps have pulled the current one into registers
      // (S_FREE), and O[g] += P(t) V(t) as soon as P(t) is published.  The whole warp walks the loop converged; one
      // elected lane issues the tcgen05 instructions.
      const int g = warp - L::kMmaWarp;
      constexpr uint32_t idesc_qk = idesc_bf16(128, HALF, 0);
      constexpr uint32_t idesc_pv = idesc_bf16(128, D, 1);
      auto issue_qk = [&](int t) {                   // S(t) = Q K(t)^T, Q read from tensor memory
        const int slot = t & (kStages - 1), k = t >> 1;
        const uint32_t sK = sRing + slot * L::kStage;
        if (k > 0) mbar_wait(bar(BAR_S_FREE + g), (k - 1) & 1);      // S(t-2) has left tensor memory
        mbar_wait(bar(BAR_FULL + slot), (t / kStages) & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t db0 = smem_desc_sw128(sK, 16, 1024);
          const uint32_t d_s = tmem + kSCol + g * kSStride;
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            // descriptor of the kk-th 16-channel slice: start address advances by 32 B inside the 128-B row, by one
            // 64-channel chunk every 4 slices (the start-address field is in 16-byte units and cannot carry out)
            const uint64_t db = db0 + (uint64_t)(((kk >> 2) * L::kKVChunk + (kk & 3) * 32) >> 4);
            mma_ts(d_s, tmem + kQCol + kk * 8, db, idesc_qk, kk > 0);
          }
          mma_commit(bar(BAR_EMPTY + slot));
          mma_commit(bar(BAR_S_FULL + g));
        }
        __syncwarp();
      };
      if (g < T) {
        mbar_wait(bar(BAR_Q_READY), 0);
        tc_fence_after();
        issue_qk(g);
        for (int t = g; t < T; t += 2) {
          if (t + 2 < T) issue_qk(t + 2);
          // O[g] += P(t) V(t)
          const int slot = t & (kStages - 1), k = t >> 1;
          const uint32_t sV = sRing + (kStages + slot) * L::kStage;
          mbar_wait(bar(BAR_FULL + kStages + slot), (t / kStages) & 1);
          mbar_wait(bar(BAR_P_FULL + g), k & 1);
          tc_fence_after();
          if (elect_one()) {
            const uint64_t db0 = smem_desc_sw128(sV, L::kKVChunk, 1024);
            const uint32_t d_o = tmem + kOCol + g * kOStride, a_p = tmem + kPCol + g * kPStride;
#pragma unroll
            for (int kk = 0; kk < HALF / 16; ++kk)
              mma_ts(d_o, a_p + kk * 8, db0 + (uint64_t)((kk * 2048) >> 4), idesc_pv, (k > 0 || kk > 0) ? 1u : 0u);
            mma_commit(bar(BAR_EMPTY + kStages + slot));
            mma_commit(bar(BAR_PV_DONE + g));
            if (t + 2 >= T) mma_commit(bar(BAR_O_FULL + g));
          }
          __syncwarp();
        }
      }
    } else {
      // =============================== softmax / lazy correction / epilogue ===============================
      // Two independent softmax groups of 4 warps: group g owns the half-tiles t = g, g+2, ... and its own O
      // accumulator, reference maximum and row sum (merged in the epilogue), so the two groups run out of phase and
      // overlap each other's MUFU bursts and TMEM / barrier latencies.  Inside a group one thread owns one query row
      // (TMEM lane) and prefetches the NEXT half-tile's S row into registers before exponentiating the current one.
      const int sw = warp & 3, g = warp >> 2;
      const uint32_t lane_base = (uint32_t)(sw * 32) << 16;
      const int row = sw * 32 + lane;                  // query row inside the tile == TMEM lane
      const bool live = row < valid_q;
      constexpr int QE = D / 2;                        // Q / O columns handled per thread in prologue / epilogue

      // ---- Q -> tensor memory (bf16 pairs, low half = even channel: the A-operand layout, same as P) ----
      {
        uint32_t qv[QE / 2];
        const uint4 *src = reinterpret_cast<const uint4 *>(p.q + b * p.q_sb + h * p.q_sh +
                                                            ((int64_t)i * BLK + row) * p.q_st + g * QE);
#pragma unroll
        for (int c = 0; c < QE / 8; ++c) {
          const uint4 v = live ? __ldg(src + c) : make_uint4(0, 0, 0, 0);
          qv[4 * c] = v.x; qv[4 * c + 1] = v.y; qv[4 * c + 2] = v.z; qv[4 * c + 3] = v.w;
        }
        const uint32_t q_addr = tmem + lane_base + kQCol + g * (QE / 2);
        if constexpr (QE / 2 == 32) tmem_st32(q_addr, *reinterpret_cast<uint32_t(*)[32]>(&qv[0]));
        else tmem_st16(q_addr, qv);
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_Q_READY));
      }

      float m_used = __int_as_float(0xff800000), l = 0.f;      // -inf / 0: a group without half-tiles merges as nothing
      int j = 0, hh = 0;
      auto advance = [&]() {
        if (hh == 0 && tile_valid(j) > HALF) hh = 1;
        else { ++j; hh = 0; }
      };
      constexpr int NLD = HALF / 32;                             // 32-column TMEM loads per S row
      auto wait_s = [&](int t) {
        mbar_wait(bar(BAR_S_FULL + g), (t >> 1) & 1);
        tc_fence_after();
      };
      auto load_s = [&](int t, int c, uint32_t (&dst)[HALF]) {   // columns [32c, 32c+32) of S(t) -> registers (no wait::ld)
        tmem_ld32(tmem + lane_base + kSCol + g * kSStride + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&dst[c * 32]));
      };
      auto release_s = [&]() {                                   // S is in registers: its TMEM buffer may be overwritten
        tc_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_S_FREE + g));
      };
      // one half-tile: `cur` holds S(t); S(t+2) is prefetched into `nxt` while P(t) is being computed
      auto step = [&](int t, uint32_t (&cur)[HALF]) {
        uint32_t (&nxt)[HALF] = cur;                     // S(t+2) is reloaded into the registers S(t) just vacated
        TR(warp, 0, t);
        const int hv = min(HALF, tile_valid(j) - hh * HALF);     // valid key columns of this half-tile (> 0)
        advance();
        if (t + 1 < T) advance();
        const int k = t >> 1;                            // this is the group's k-th half-tile
        if (hv < HALF) {                                         // padded key columns -> -inf (warp-uniform branch)
#pragma unroll
          for (int c = 0; c < HALF; ++c) if (c >= hv) cur[c] = 0xff800000u;
        }
        float mx0 = __uint_as_float(cur[0]), mx1 = __uint_as_float(cur[1]), mx2 = __uint_as_float(cur[2]), mx3 = __uint_as_float(cur[3]);
#pragma unroll
        for (int c = 4; c < HALF; c += 4) {
          mx0 = fmaxf(mx0, __uint_as_float(cur[c]));
          mx1 = fmaxf(mx1, __uint_as_float(cur[c + 1]));
          mx2 = fmaxf(mx2, __uint_as_float(cur[c + 2]));
          mx3 = fmaxf(mx3, __uint_as_float(cur[c + 3]));
        }
        const float m_new = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * p.scale_log2;
        TR(warp, 2, t);

        // lazy rescale: the reference maximum only moves when the row maximum grew by more than 2^8
        bool need = false;
        if (t < 2) m_used = m_new;
        else need = m_new > m_used + kRescaleThreshold;
        if (__ballot_sync(0xffffffffu, need)) {
          // this group's O is being accumulated by PV(t-2), which commits to PV_DONE[g] as its use number (t-2)/2;
          // PV(t-4) is known complete (S(t) exists), so the parity test is unambiguous
          mbar_wait(bar(BAR_PV_DONE + g), (k - 1) & 1);
          tc_fence_after();
          const float f = need ? ex2_approx(m_used - m_new) : 1.0f;
          if (need) { m_used = m_new; l *= f; }
#pragma unroll 1
          for (int c = 0; c < D / 16; ++c) {             // rare path: small chunks keep the register footprint low
            uint32_t o[16];
            const uint32_t o_addr = tmem + lane_base + kOCol + g * kOStride + c * 16;
            tmem_ld16(o_addr, o);
            tc_wait_ld();
#pragma unroll
            for (int e = 0; e < 16; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * f);
            tmem_st16(o_addr, o);
          }
          tc_wait_st();
        }

        // P = exp2(s*scale - m_used), row sum in fp32, bf16 pairs packed low = even column.  kEmuOf4 of every 4
        // column pairs take the FMA-pipe exp2 (li_ptx.cuh), the others the MUFU.  The next half-tile of this group,
        // S(t+2), is prefetched into registers chunk by chunk as the registers of S(t) die, so that its TMEM latency
        // hides behind the exponentials without doubling the register footprint.
        const uint64_t sc2 = pack2(p.scale_log2, p.scale_log2), nm2 = pack2(-m_used, -m_used);
        uint64_t sum_a = pack2(0.f, 0.f), sum_b = pack2(0.f, 0.f);
        uint32_t pk[HALF / 2];
        const bool more = t + 2 < T;
#pragma unroll
        for (int ch = 0; ch < NLD; ++ch) {
#pragma unroll
          for (int c = ch * 16; c < ch * 16 + 16; ++c) {
            const uint64_t x2 = fma2(pack2(__uint_as_float(cur[2 * c]), __uint_as_float(cur[2 * c + 1])), sc2, nm2);
            float p0, p1;
            if ((c & 3) < kEmuOf4) {
              exp2_emulated2(x2, p0, p1);
            } else {
              float x0, x1;
              unpack2(x2, x0, x1);
              p0 = ex2_approx(x0);
              p1 = ex2_approx(x1);
            }
            if (c & 1) sum_b = add2(sum_b, pack2(p0, p1));
            else sum_a = add2(sum_a, pack2(p0, p1));
            pk[c] = pack_bf16x2(p0, p1);
          }
          if (kEarlyPrefetch && ch == 0 && more) {
            wait_s(t + 2);
            load_s(t + 2, 0, nxt);
          }
        }
        {
          float a0, a1;
          unpack2(add2(sum_a, sum_b), a0, a1);
          l += a0 + a1;
        }
        TR(warp, 5, t);
        // P(t) goes to the group's own P columns, which PV(t-2) must have finished reading
        if (k > 0) {
          mbar_wait(bar(BAR_PV_DONE + g), (k - 1) & 1);
          tc_fence_after();
        }
        const uint32_t p_addr = tmem + lane_base + kPCol + g * kPStride;
        if constexpr (HALF == 64) tmem_st32(p_addr, *reinterpret_cast<uint32_t(*)[32]>(&pk[0]));
        else tmem_st16(p_addr, pk);
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_P_FULL + g));
        TR(warp, 7, t);
        if (more) {
          if (!kEarlyPrefetch) { wait_s(t + 2); load_s(t + 2, 0, nxt); }
          if (NLD == 2) load_s(t + 2, 1, nxt);
          release_s();                                   // S(t+2) row is now in registers
        }
        TR(warp, 8, t);
      };

      {
        uint32_t sa[HALF];
        if (g < T) {
          if (g == 1) advance();                         // group 1 starts at half-tile 1
          if (g == 1 && kStaggerCycles > 0) {
            // start the second group half a step late: two groups in phase would fight for the MUFU during their
            // exponentials and leave it idle during their other phases
            const long long t_start = clock64();
            while (clock64() - t_start < kStaggerCycles) {
            }
          }
          wait_s(g);
#pragma unroll
          for (int c = 0; c < NLD; ++c) load_s(g, c, sa);
          release_s();
          for (int t = g; t < T; t += 2) step(t, sa);
        }
      }

      // ---- epilogue: merge the two groups' partial results, O / l -> bf16 in linear token order (no untile pass).
      //      Thread (g, row) stores columns [g*D/2, (g+1)*D/2) of its row. ----
      sXch[(g * 2 + 0) * 128 + row] = m_used;
      sXch[(g * 2 + 1) * 128 + row] = l;
      named_bar_sync(1 + sw, 64);
      const float m_o = sXch[((g ^ 1) * 2 + 0) * 128 + row], l_o = sXch[((g ^ 1) * 2 + 1) * 128 + row];
      const float m_all = fmaxf(m_used, m_o);
      const float w_me = ex2_approx(m_used - m_all), w_o = ex2_approx(m_o - m_all);   // 2^-inf = 0 for an idle group
      const float l_all = l * w_me + l_o * w_o;
      const float wA = (g == 0 ? w_me : w_o) / l_all, wB = (g == 0 ? w_o : w_me) / l_all;
      const bool hasB = T > 1;
      mbar_wait(bar(BAR_O_FULL), 0);
      if (hasB) mbar_wait(bar(BAR_O_FULL1), 0);
      tc_fence_after();
      uint16_t *orow = p.o + (((int64_t)b * p.H + h) * p.Lq + (int64_t)i * BLK + row) * D + g * QE;
#pragma unroll
      for (int c = 0; c < QE / 16; ++c) {
        uint32_t oa[16], ob[16];
        tmem_ld16(tmem + lane_base + kOCol + g * QE + c * 16, oa);
        if (hasB) tmem_ld16(tmem + lane_base + kOCol + kOStride + g * QE + c * 16, ob);
        tc_wait_ld();
        float r[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
          r[e] = __uint_as_float(oa[e]) * wA;
          if (hasB) r[e] = fmaf(__uint_as_float(ob[e]), wB, r[e]);
        }
        if (live) {
#pragma unroll
          for (int e = 0; e < 16; e += 8) {
            uint4 v;
            v.x = pack_bf16x2(r[e + 0], r[e + 1]);
            v.y = pack_bf16x2(r[e + 2], r[e + 3]);
            v.z = pack_bf16x2(r[e + 4], r[e + 5]);
            v.w = pack_bf16x2(r[e + 6], r[e + 7]);
            *reinterpret_cast<uint4 *>(orow + c * 16 + e) = v;
          }
        }
      }
      if (g == 0 && live && p.lse != nullptr)
        p.lse[((int64_t)b * p.H + h) * p.Lq + (int64_t)i * BLK + row] = (m_all + log2f(l_all)) * 0.6931471805599453f;
    }
  } else {
    // empty context: o = 0, lse = -inf
    if (warp < 4) {
      const int row = warp * 32 + lane;
      if (row < valid_q) {
        uint16_t *orow = p.o + (((int64_t)b * p.H + h) * p.Lq + (int64_t)i * BLK + row) * D;
        for (int c = 0; c < D; c += 8) *reinterpret_cast<uint4 *>(orow + c) = make_uint4(0, 0, 0, 0);
        if (p.lse != nullptr) p.lse[((int64_t)b * p.H + h) * p.Lq + (int64_t)i * BLK + row] = __int_as_float(0xff800000);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == L::kMmaWarp) tmem_dealloc(tmem, kTmemCols);
}

template <int D, int BLK>
static int launch_one(const AttnParams &ap, const BatchMeta &meta, const CUtensorMap &tm_k_full, const CUtensorMap &tm_k_8,
                      const CUtensorMap &tm_v_full, const CUtensorMap &tm_v_8, cudaStream_t st) {
  auto kern = li_sparse_attn_kernel<D, BLK>;
  constexpr int smem = AttnCfg<D, BLK>::kTotal;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return (int)e;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(ap.Nqb, ap.H, ap.B);
  cfg.blockDim = dim3(AttnCfg<D, BLK>::kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  e = cudaLaunchKernelEx(&cfg, kern, ap, meta, tm_k_full, tm_k_8, tm_v_full, tm_v_8);
  return (int)e;
}

int launch_attn(const AttnParams &ap, const BatchMeta &meta, int d, int blk, const CUtensorMap &tm_k_full,
                const CUtensorMap &tm_k_8, const CUtensorMap &tm_v_full, const CUtensorMap &tm_v_8, cudaStream_t st,
                int64_t *n_launches) {
  int e;
  if (d == 128 && blk == 128) e = launch_one<128, 128>(ap, meta, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st);
  else if (d == 128 && blk == 64) e = launch_one<128, 64>(ap, meta, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st);
  else if (d == 64 && blk == 128) e = launch_one<64, 128>(ap, meta, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st);
  else e = launch_one<64, 64>(ap, meta, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st);
  if (e == 0 && n_launches) *n_launches += 1;
  return e;
}

}  // namespace li
