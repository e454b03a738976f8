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

constexpr int kSelCap = 1024;       // selected-block indices staged in shared memory (rest read from global)
constexpr int kTmemCols = 512;
constexpr int kQCol = 0, kSCol = 64, kSStride = 64, kOCol = 256;
constexpr int kStages = 8;          // K/V half-tile ring
constexpr int kSBufs = 3;
constexpr float kRescaleThreshold = 8.0f;   // log2 units: P stays <= 2^8 between lazy rescales
#ifndef LI_EMU_OF_4
#define LI_EMU_OF_4 0
#endif
constexpr int kEmuOf4 = LI_EMU_OF_4;        // of every 4 column pairs, how many use the FMA-pipe exp2

template <int D, int BLK>
struct AttnCfg {
  static constexpr int HALF = BLK / 2;
  static constexpr int CW = 16;                        // S columns per softmax thread per half-tile
  static constexpr int NPART = HALF / CW;              // threads per query row (4 for BLK=128, 2 for BLK=64)
  static constexpr int kSoftmaxWarps = 4 * NPART;
  static constexpr int kProducerWarp = kSoftmaxWarps, kMmaWarp = kSoftmaxWarps + 1;
  static constexpr int kThreads = (kSoftmaxWarps + 2) * 32;
  static constexpr int kKVChunk = HALF * 128;          // bytes of one 64-column chunk of a K or V half-tile
  static constexpr int kStage = (D / 64) * kKVChunk;
  static constexpr int kOffRing = 0;
  static constexpr int kOffSel = kStages * kStage;
  static constexpr int kOffXch = kOffSel + kSelCap * 4;              // row-max / row-sum exchange: [3][NPART][128] floats
  static constexpr int kOffBar = kOffXch + 3 * NPART * 128 * 4;
  static constexpr int kTotal = kOffBar + 512 + 1024;                // + barriers + slack for 1024-B alignment
};

enum {
  BAR_FULL = 0,                        // +slot
  BAR_EMPTY = BAR_FULL + kStages,      // +slot
  BAR_S_FULL = BAR_EMPTY + kStages,    // +buffer
  BAR_P_FULL = BAR_S_FULL + kSBufs,    // +buffer
  BAR_PV_DONE = BAR_P_FULL + kSBufs,   // +(t & 1)
  BAR_Q_READY = BAR_PV_DONE + 2,
  BAR_O_FULL,
  BAR_COUNT
};

template <int D, int BLK>
__global__ void __launch_bounds__(AttnCfg<D, BLK>::kThreads, 1)
li_sparse_attn_kernel(const AttnParams p, const BatchMeta meta, const __grid_constant__ CUtensorMap tm_k_full,
                      const __grid_constant__ CUtensorMap tm_k_8, const __grid_constant__ CUtensorMap tm_v_full,
                      const __grid_constant__ CUtensorMap tm_v_8) {
  using L = AttnCfg<D, BLK>;
  constexpr int HALF = L::HALF, CW = L::CW, NPART = L::NPART;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *smem = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t sRing = smem_base + L::kOffRing;
  int32_t *sSel = reinterpret_cast<int32_t *>(smem + L::kOffSel);
  volatile float *sXch = reinterpret_cast<volatile float *>(smem + L::kOffXch);
  const uint32_t bar0 = smem_base + L::kOffBar;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + L::kOffBar + 8 * BAR_COUNT);
  auto bar = [&](int i) { return bar0 + 8u * i; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z;

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
  if (warp == L::kProducerWarp && lane == 0) {
    tma_prefetch_desc(&tm_k_full);
    tma_prefetch_desc(&tm_v_full);
    tma_prefetch_desc(&tm_k_8);
    tma_prefetch_desc(&tm_v_8);
    for (int k = 0; k < BAR_COUNT; ++k) {
      const bool by_softmax = (k >= BAR_P_FULL && k < BAR_P_FULL + kSBufs) || k == BAR_Q_READY;
      mbar_init(bar(k), by_softmax ? L::kSoftmaxWarps : 1);
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
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  auto sel_at = [&](int jj) -> int { return jj < kSelCap ? sSel[jj] : sel_row[jj]; };
  // valid key columns of attended tile j (chunk blocks first, then the selected historical blocks)
  auto tile_valid = [&](int j) -> int {
    if (j < Nc) return j == Nc - 1 ? tail_cur : BLK;
    return sel_at(j - Nc) == M - 1 ? tail_hist : BLK;
  };
  // number of half-tiles with at least one valid key (a half-tile without any is skipped by every role)
  int T = 2 * n_tiles;
  if (Nc > 0 && tail_cur <= HALF) --T;
  if (cnt > 0 && sel_at(cnt - 1) == M - 1 && tail_hist <= HALF) --T;

  if (T > 0) {
    if (warp == L::kProducerWarp) {
      // =============================== TMA producer ===============================
      if (lane == 0) {
        int n = 0;                                   // running load index: slot = n % kStages
        // loads HALF rows [t0, t0+HALF) of a region (history or chunk) into the next ring slot
        auto load_half = [&](const CUtensorMap *tm_full, const CUtensorMap *tm_8, int j, int hh) {
          const bool is_cur = j < Nc;
          const int blk = is_cur ? j : sel_at(j - Nc);
          const int32_t *pages = p.frame_idx + foff + (is_cur ? n_hist : 0);
          const int region_len = is_cur ? L_cur : L_hist;
          const int t0 = blk * BLK + hh * HALF;
          const int slot = n & (kStages - 1);
          const uint32_t dst = sRing + slot * L::kStage, mb = bar(BAR_FULL + slot);
          mbar_wait(bar(BAR_EMPTY + slot), ((n / kStages) & 1) ^ 1);
          mbar_arrive_expect_tx(mb, HALF * D * 2);
          const int t_last = min(t0 + HALF, region_len) - 1;
          const int pg0 = t0 / p.T_f;
          if (p.has_box_full && pg0 == t_last / p.T_f) {
            // inside one page: one box per 64-column chunk; rows past the page end are zero-filled by the
            // hardware (a region always ends on a page boundary)
            const int page = pages[pg0];
            const int row = t0 - pg0 * p.T_f;
#pragma unroll
            for (int c = 0; c < D / 64; ++c) tma_load_4d(dst + c * L::kKVChunk, tm_full, mb, c * 64, row, h, page);
          } else {
            // straddles frames: 8-row pieces (one SWIZZLE_128B atom each, destinations stay 1024-B aligned)
            int cur_pg = -1, page = 0;
            for (int g = 0; g < HALF / 8; ++g) {
              const int t = t0 + g * 8;
              int row = p.T_f;             // out of bounds -> zeros
              if (t < region_len) {
                const int pg = t / p.T_f;
                if (pg != cur_pg) { cur_pg = pg; page = pages[pg]; }
                row = t - pg * p.T_f;
              }
#pragma unroll
              for (int c = 0; c < D / 64; ++c)
                tma_load_4d(dst + c * L::kKVChunk + g * 1024, tm_8, mb, c * 64, row, h, page);
            }
          }
          ++n;
        };
        auto advance = [&](int &j, int &hh) {
          if (hh == 0 && tile_valid(j) > HALF) hh = 1;
          else { ++j; hh = 0; }
        };

        // load order == consumption order of the MMA warp: K0 K1 K2 | V0 K3 | V1 K4 | ...
        int kj = 0, kh = 0, vj = 0, vh = 0;
        for (int t = 0; t < kSBufs && t < T; ++t) { load_half(&tm_k_full, &tm_k_8, kj, kh); advance(kj, kh); }
        for (int t = 0; t < T; ++t) {
          load_half(&tm_v_full, &tm_v_8, vj, vh); advance(vj, vh);
          if (t + kSBufs < T) { load_half(&tm_k_full, &tm_k_8, kj, kh); advance(kj, kh); }
        }
      }
    } else if (warp == L::kMmaWarp) {
      // =============================== MMA issuer ===============================
      if (lane == 0) {
        constexpr uint32_t idesc_qk = idesc_bf16(128, HALF, 0);
        constexpr uint32_t idesc_pv = idesc_bf16(128, D, 1);
        int c = 0;                                   // running consume index: slot = c % kStages
        auto issue_qk = [&](int t) {                 // S(t) = Q K(t)^T, Q read from tensor memory
          const int slot = c & (kStages - 1);
          const uint32_t sK = sRing + slot * L::kStage;
          mbar_wait(bar(BAR_FULL + slot), (c / kStages) & 1);
          tc_fence_after();
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            const uint64_t db = smem_desc_sw128(sK + (kk >> 2) * L::kKVChunk + (kk & 3) * 32, 16, 1024);
            mma_ts(tmem + kSCol + (t % kSBufs) * kSStride, tmem + kQCol + kk * 8, db, idesc_qk, kk > 0);
          }
          mma_commit(bar(BAR_EMPTY + slot));
          mma_commit(bar(BAR_S_FULL + (t % kSBufs)));
          ++c;
        };
        mbar_wait(bar(BAR_Q_READY), 0);
        tc_fence_after();
        for (int t = 0; t < kSBufs && t < T; ++t) issue_qk(t);
        for (int t = 0; t < T; ++t) {
          // O += P(t) V(t)
          const int slot = c & (kStages - 1);
          const uint32_t sV = sRing + slot * L::kStage;
          mbar_wait(bar(BAR_FULL + slot), (c / kStages) & 1);
          mbar_wait(bar(BAR_P_FULL + (t % kSBufs)), (t / kSBufs) & 1);
          tc_fence_after();
#pragma unroll
          for (int kk = 0; kk < HALF / 16; ++kk) {
            const uint64_t db = smem_desc_sw128(sV + kk * 2048, L::kKVChunk, 1024);
            mma_ts(tmem + kOCol, tmem + kSCol + (t % kSBufs) * kSStride + kk * 8, db, idesc_pv, (t > 0 || kk > 0) ? 1u : 0u);
          }
          mma_commit(bar(BAR_EMPTY + slot));
          mma_commit(bar(BAR_PV_DONE + (t & 1)));
          if (t == T - 1) mma_commit(bar(BAR_O_FULL));
          ++c;
          if (t + kSBufs < T) issue_qk(t + kSBufs);
        }
      }
      __syncwarp();
    } else {
      // =============================== softmax / lazy correction / epilogue ===============================
      // NPART threads per query row: warps w, w+4, ... own the same TMEM lanes 32(w%4).. and split every half-tile's
      // columns (and Q's / O's columns) among them.  They agree on the row maximum through shared memory and a named
      // barrier; each keeps a partial row sum.
      const int sw = warp & 3, part = warp >> 2;
      const uint32_t lane_base = (uint32_t)(sw * 32) << 16;
      const int row = sw * 32 + lane;                  // query row inside the tile == TMEM lane
      const bool live = row < valid_q;
      constexpr int QE = D / NPART;                    // Q / O elements (columns of O) per thread

      // ---- Q -> tensor memory (bf16 pairs, low half = even channel: the A-operand layout, same as P) ----
      {
        uint32_t qv[QE / 2];
        const uint4 *src = reinterpret_cast<const uint4 *>(p.q + b * p.q_sb + h * p.q_sh +
                                                            ((int64_t)i * BLK + row) * p.q_st + part * QE);
#pragma unroll
        for (int c = 0; c < QE / 8; ++c) {
          const uint4 v = live ? __ldg(src + c) : make_uint4(0, 0, 0, 0);
          qv[4 * c] = v.x; qv[4 * c + 1] = v.y; qv[4 * c + 2] = v.z; qv[4 * c + 3] = v.w;
        }
        const uint32_t q_addr = tmem + lane_base + kQCol + part * (QE / 2);
        if constexpr (QE / 2 == 32) tmem_st32(q_addr, *reinterpret_cast<uint32_t(*)[32]>(&qv[0]));
        else if constexpr (QE / 2 == 16) tmem_st16(q_addr, qv);
        else tmem_st8(q_addr, qv);
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_Q_READY));
      }

      float m_used = 0.f, l = 0.f;
      int j = 0, hh = 0;
      for (int t = 0; t < T; ++t) {
        const int tv = tile_valid(j);
        const int hv = min(HALF, tv - hh * HALF) - part * CW;   // valid columns among this thread's CW (may be <= 0)
        if (hh == 0 && tv > HALF) hh = 1;
        else { ++j; hh = 0; }
        const int u = t % kSBufs;
        const uint32_t s_addr = tmem + lane_base + kSCol + u * kSStride;

        mbar_wait(bar(BAR_S_FULL + u), (t / kSBufs) & 1);
        tc_fence_after();
        uint32_t s[CW];
        tmem_ld16(s_addr + part * CW, s);
        tc_wait_ld();
        if (hv < CW) {                                 // padded key columns -> -inf (warp-uniform branch)
#pragma unroll
          for (int c = 0; c < CW; ++c) if (c >= hv) s[c] = 0xff800000u;
        }
        float mx0 = __uint_as_float(s[0]), mx1 = __uint_as_float(s[1]), mx2 = __uint_as_float(s[2]), mx3 = __uint_as_float(s[3]);
#pragma unroll
        for (int c = 4; c < CW; c += 4) {
          mx0 = fmaxf(mx0, __uint_as_float(s[c]));
          mx1 = fmaxf(mx1, __uint_as_float(s[c + 1]));
          mx2 = fmaxf(mx2, __uint_as_float(s[c + 2]));
          mx3 = fmaxf(mx3, __uint_as_float(s[c + 3]));
        }
        float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
        sXch[(u * NPART + part) * 128 + row] = mx;
        named_bar_sync(1 + sw, NPART * 32);
#pragma unroll
        for (int q = 0; q < NPART; ++q) mx = fmaxf(mx, sXch[(u * NPART + q) * 128 + row]);
        const float m_new = mx * p.scale_log2;

        // lazy rescale: the reference maximum only moves when the row maximum grew by more than 2^8
        bool need = false;
        if (t == 0) m_used = m_new;
        else need = m_new > m_used + kRescaleThreshold;
        if (__ballot_sync(0xffffffffu, need)) {
          // O is being accumulated by PV(t-1): wait for it.  PV(t) commits to barrier t&1, so the parity of use
          // (t-1)/2 of barrier (t-1)&1 is unambiguous.  All threads of a row take this branch together (same m_new);
          // each rescales its own columns of O.
          mbar_wait(bar(BAR_PV_DONE + ((t - 1) & 1)), ((t - 1) >> 1) & 1);
          tc_fence_after();
          const float f = need ? ex2_approx(m_used - m_new) : 1.0f;
          if (need) { m_used = m_new; l *= f; }
#pragma unroll 1
          for (int c = 0; c < QE / 16; ++c) {            // rare path: small chunks keep the register footprint low
            uint32_t o[16];
            const uint32_t o_addr = tmem + lane_base + kOCol + part * QE + c * 16;
            tmem_ld16(o_addr, o);
            tc_wait_ld();
#pragma unroll
            for (int e = 0; e < 16; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * f);
            tmem_st16(o_addr, o);
          }
        }

        // P = exp2(s*scale - m_used), row sum in fp32, bf16 pairs packed low = even column.  kEmuOf4 of every 4
        // column pairs take the FMA-pipe exp2 (li_ptx.cuh), the others the MUFU.
        const uint64_t sc2 = pack2(p.scale_log2, p.scale_log2), nm2 = pack2(-m_used, -m_used);
        uint64_t sum_a = pack2(0.f, 0.f), sum_b = pack2(0.f, 0.f);
        uint32_t pk[CW / 2];
#pragma unroll
        for (int c = 0; c < CW / 2; ++c) {
          const uint64_t x2 = fma2(pack2(__uint_as_float(s[2 * c]), __uint_as_float(s[2 * c + 1])), sc2, nm2);
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
        {
          float a0, a1;
          unpack2(add2(sum_a, sum_b), a0, a1);
          l += a0 + a1;
        }
        tmem_st8(s_addr + part * (CW / 2), pk);
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_P_FULL + u));
      }

      // epilogue: O / l -> bf16, stored in linear token order (no untile pass); each thread stores its QE columns
      {
        const int xb = T % kSBufs;                     // exchange buffer not used by the last half-tile
        sXch[(xb * NPART + part) * 128 + row] = l;
        named_bar_sync(1 + sw, NPART * 32);
        l = 0.f;
#pragma unroll
        for (int q = 0; q < NPART; ++q) l += sXch[(xb * NPART + q) * 128 + row];
      }
      mbar_wait(bar(BAR_O_FULL), 0);
      tc_fence_after();
      const float inv_l = 1.0f / l;
      uint16_t *orow = p.o + (((int64_t)b * p.H + h) * p.Lq + (int64_t)i * BLK + row) * D + part * QE;
#pragma unroll
      for (int c = 0; c < QE / 16; ++c) {
        uint32_t o[16];
        tmem_ld16(tmem + lane_base + kOCol + part * QE + c * 16, o);
        tc_wait_ld();
        if (live) {
#pragma unroll
          for (int e = 0; e < 16; e += 8) {
            uint4 v;
            v.x = pack_bf16x2(__uint_as_float(o[e + 0]) * inv_l, __uint_as_float(o[e + 1]) * inv_l);
            v.y = pack_bf16x2(__uint_as_float(o[e + 2]) * inv_l, __uint_as_float(o[e + 3]) * inv_l);
            v.z = pack_bf16x2(__uint_as_float(o[e + 4]) * inv_l, __uint_as_float(o[e + 5]) * inv_l);
            v.w = pack_bf16x2(__uint_as_float(o[e + 6]) * inv_l, __uint_as_float(o[e + 7]) * inv_l);
            *reinterpret_cast<uint4 *>(orow + c * 16 + e) = v;
          }
        }
      }
      if (part == 0 && live && p.lse != nullptr)
        p.lse[((int64_t)b * p.H + h) * p.Lq + (int64_t)i * BLK + row] = (m_used + log2f(l)) * 0.6931471805599453f;
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
