// li_attn.cu -- li_sparse_attn for sm_100a: block-sparse flash attention over C_i = K^curr U S_i
// (Eq. 11), K/V tiles fetched IN PLACE from the frame-paged cache by TMA with the page
// as a tensor coordinate (replaces the paper's KV-Prep / Untile-Scatter copies).
//
// One CTA = one query block (BLK query rows, padded to the 128-row UMMA tile) of one (call, head); two CTAs per SM
// (256 TMEM columns and ~101 KB of shared memory each), whose pipelines overlap each other's latencies.
// Every attended KV block is processed as two HALF-tiles of HALF = BLK/2 keys, software-pipelined inside the CTA:
// S is double-buffered in TMEM, so the tensor core computes S(t+1) = Q K(t+1)^T while the softmax warps work on
// S(t), and O += P(t) V(t) is issued as soon as P(t) is written.  Tensor-core issue order:
//     QK(0) QK(1) | PV(0) QK(2) | PV(1) QK(3) | ...      (K/V half-tiles are loaded in exactly this order
//                                                         into a 4-slot shared-memory ring)
//   warps 0-3 : softmax + lazy correction + epilogue; warp w owns TMEM lanes 32w..32w+31 (one query row per thread)
//   warp 4    : TMA producer: Q once, then the K/V half-tiles.  The warp stays converged, an elected lane issues;
//               the call's frame list is staged in shared memory (a global load per tile would pace the pipeline)
//   warp 5    : TMEM allocation and the tcgen05.mma issuer (converged warp, elected lane, descriptors by addition)
// TMEM (256 columns): [0,HALF) S_a, [64,64+HALF) S_b (fp32; P in bf16 overlays the first HALF/2 columns of its S
// buffer once S has been read), [128,128+D) O.
// On B200 this kernel runs into the 1 kW power cap (SM clock ~1.6 GHz under load); DESIGN.md section 6.3 lists the
// measured alternatives (one CTA per SM with Q in tensor memory, two softmax groups, FMA-pipe exp2, full-tile QK,
// speculative / prefetching softmax loop, ...).  The TMEM budget above is what fixes the design: the one measured
// gain left (QK with Q as a tensor-memory A operand, -5.7 %) needs 64 more columns than two co-resident CTAs have.
// KV8 instances (LI_FLAG_KV_FP8): K/V pages hold e4m3 codes; the softmax warps first turn the bf16 Q
// tile into its per-row e4m3 image in shared memory, both contractions run on tcgen05.mma.kind::f8f6f4 and P is
// rounded to e4m3 (four keys per TMEM column).
#include <atomic>

#include "li_internal.h"
#include "li_ptx.cuh"

namespace li {

constexpr int kInfoCap = 2048;      // attended tiles whose 3-D geometry is tabulated in shared memory
constexpr int kPageCap = 256;       // frame-list entries staged in shared memory (rest read from global)
constexpr int kSelCap = 1024;       // selected-block indices staged in shared memory (rest read from global)
constexpr int kTmemCols = 256;
constexpr int kSbCol = 64;
constexpr int kOCol = 128;
constexpr int kStages = 4;
constexpr float kRescaleThreshold = 8.0f;   // log2 units: P stays <= 2^8 between lazy rescales
#ifndef LI_EMU_OF_4
#define LI_EMU_OF_4 0
#endif
constexpr int kEmuOf4 = LI_EMU_OF_4;        // of every 4 column pairs, how many use the FMA-pipe exp2

template <int D, int BLK, bool KV8 = false>
struct AttnSmem {
  static constexpr int HALF = BLK / 2;
  static constexpr int kQChunk = 128 * 128;            // bytes of one 64-column chunk of the 128-row (bf16) Q tile
  static constexpr int kKVChunk = HALF * 128;          // bytes of one 128-byte-wide chunk of a K or V half-tile
  static constexpr int kKVChunks = KV8 ? D / 128 : D / 64;   // 128 bytes = 64 bf16 channels or 128 e4m3 channels
  static constexpr int kQ = (D / 64) * kQChunk;
  static constexpr int kQ8 = KV8 ? 128 * 128 : 0;      // FP8 pages: the e4m3 image of the Q tile (128 rows x 128 bytes)
  static constexpr int kStage = kKVChunks * kKVChunk;
  static constexpr int kOffQ = 0;
  static constexpr int kOffQ8 = kQ;
  static constexpr int kOffRing = kQ + kQ8;
  static constexpr int kOffSel = kOffRing + kStages * kStage;
  static constexpr int kOffPages = kOffSel + kSelCap * 4;   // this call's frame list, staged once
  static constexpr int kOffInfo = kOffPages + kPageCap * 4;  // 3-D: per attended tile (frames present) | (valid rows per slice) << 8
  static constexpr int kOffBar = kOffInfo + kInfoCap * 2;
  static constexpr int kTotal = kOffBar + 256 + 1024;  // + barriers + slack for 1024-B alignment
};

enum {
  BAR_Q_FULL = 0,
  BAR_FULL = 1,                    // +slot
  BAR_EMPTY = BAR_FULL + kStages,  // +slot
  BAR_S_FULL = BAR_EMPTY + kStages,  // +buffer
  BAR_P_FULL = BAR_S_FULL + 2,       // +buffer
  BAR_PV_DONE = BAR_P_FULL + 2,
  BAR_O_FULL,
  BAR_Q8,                            // FP8 pages: the softmax warps have written the e4m3 image of Q
  BAR_COUNT
};

// n / dv for n, dv < 65536 by a multiply-high with mg = floor(2^32 / dv) + 1 (exact there: n * dv < 2^32)
__device__ __forceinline__ int div_magic(int n, int dv, uint32_t mg) {
  return (n | dv) < 65536 ? (int)__umulhi((uint32_t)n, mg) : n / dv;
}

// -inf into the key columns c of a half-tile with (c mod 32) >= V (compile-time positions: V..31 of every 32-row slice)
template <int V, int HALF>
__device__ __forceinline__ void mask_slice_tail(uint32_t (&s)[HALF]) {
#pragma unroll
  for (int c = 0; c < HALF; ++c)
    if ((c & 31) >= V) s[c] = 0xff800000u;
}

// linear token of query row `row` of query block i, or -1 for a padding row ("masked stores")
template <int BLK, bool K3D>
__device__ __forceinline__ int64_t row_token(const AttnParams &p, int i, int row) {
  if (K3D) {
    const Tiling &tl = p.tl;
    const int per = tl.Hb * tl.Wb, tg = i / per, hb = (i - tg * per) / tl.Wb, wb = i - tg * per - hb * tl.Wb;
    const int f = tg * tl.bt + (row >> 5), within = row & 31, y = hb * tl.bh + within / tl.bw, x = wb * tl.bw + within % tl.bw;
    return (row < BLK && f < p.Lq / p.T_f && y < tl.gh && x < tl.gw) ? (int64_t)f * p.T_f + y * tl.gw + x : -1;
  }
  return row < min(BLK, p.Lq - i * BLK) ? (int64_t)i * BLK + row : -1;
}

template <int D, int BLK, bool K3D, bool TEXT, bool SPLIT, bool KV8>
__device__ __forceinline__ void attn_body(const AttnParams &p, const BatchMeta &meta, const CUtensorMap &tm_q,
                                          const CUtensorMap &tm_k_full, const CUtensorMap &tm_k_8,
                                          const CUtensorMap &tm_v_full, const CUtensorMap &tm_v_8,
                                          const CUtensorMap &tm_tk, const CUtensorMap &tm_tv) {
  using L = AttnSmem<D, BLK, KV8>;
  constexpr int HALF = L::HALF;
  constexpr int KCH = L::kKVChunks, CW = KV8 ? 128 : 64;   // K/V chunks per half-tile, channels per chunk
  constexpr int EB = KV8 ? 1 : 2;                          // bytes per K/V element
  static_assert(!KV8 || (D == 128 && !TEXT), "FP8 pages: d = 128, no text prefix");
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *smem = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t sQ = smem_base + L::kOffQ, sRing = smem_base + L::kOffRing;
  int32_t *sSel = reinterpret_cast<int32_t *>(smem + L::kOffSel);
  int32_t *sPages = reinterpret_cast<int32_t *>(smem + L::kOffPages);
  uint16_t *sInfo = reinterpret_cast<uint16_t *>(smem + L::kOffInfo);
  const uint32_t bar0 = smem_base + L::kOffBar;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + L::kOffBar + 8 * BAR_COUNT);
  int *sT = reinterpret_cast<int *>(smem + L::kOffBar + 8 * BAR_COUNT + 8);   // half-tile count (3-D mode)
  int *sTailPos = sT + 1;                              // 1-D: position of the partial history tail block in the row's list
  auto bar = [&](int i) { return bar0 + 8u * i; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // CTA -> (query block i, head h, call b) and, in the tail wave, which of n_split ranges of its half-tiles
  // (SPLIT launches use a linear grid; the others the grid (Nqb, H, B) and none of this code)
  int work = blockIdx.x, sq = 0, ns = 1;
  if (SPLIT && work >= p.split_first) {
    const int e = work - p.split_first;
    work = p.split_first + e / p.n_split;
    sq = e % p.n_split;
    ns = p.n_split;
  }
  const int i = SPLIT ? work % p.Nqb : blockIdx.x, h = SPLIT ? (work / p.Nqb) % p.H : blockIdx.y,
            b = SPLIT ? work / (p.Nqb * p.H) : blockIdx.z;

  // ---- per-tile integer bookkeeping (Eq. 11 context assembly) ----
  const int foff = meta.frame_off[b];
  const int n_frames = meta.frame_off[b + 1] - foff;
  const int n_hist = n_frames - p.n_cur;
  const int L_hist = n_hist * p.T_f;
  const int L_cur = p.n_cur * p.T_f;
  const Tiling tl = p.tl;
  constexpr bool k3d = K3D;                            // 3-D blocks: BLK = bt*32, 32 = bh*bw rows per frame slice
  constexpr int SPH = HALF / 32;                       // 32-row slices per half-tile
  const int per = tl.Hb * tl.Wb;                       // blocks per temporal group (3-D)
  // block index -> (temporal group, row block, column block)
  auto split3 = [&](int blk, int &tg, int &hb, int &wb) {
    tg = blk / per;
    const int r = blk - tg * per;
    hb = r / tl.Wb;
    wb = r - hb * tl.Wb;
  };
  const int M = tl.num_blocks(n_hist, p.T_f, BLK);
  const int Nc = tl.num_blocks(p.n_cur, p.T_f, BLK);
  const int n_qf = p.Lq / p.T_f;                       // query frames (3-D)
  const int Nt = TEXT ? (p.Lt + BLK - 1) / BLK : 0;    // text tiles (T of Eq. 11): dense, attended first, 1-D
  const int tail_text = p.Lt - (Nt - 1) * BLK;
  const int64_t row_id = ((int64_t)b * p.H + h) * p.Nqb + i;
  const int tail_cur = L_cur - (Nc - 1) * BLK, tail_hist = L_hist - (M - 1) * BLK;

  // ---- one-time setup (independent of the previous kernel: overlaps its tail under PDL) ----
  if (warp == 4 && lane == 0) {
    tma_prefetch_desc(&tm_q);
    tma_prefetch_desc(&tm_k_full);
    tma_prefetch_desc(&tm_v_full);
    tma_prefetch_desc(&tm_k_8);
    tma_prefetch_desc(&tm_v_8);
    if (TEXT) {
      tma_prefetch_desc(&tm_tk);
      tma_prefetch_desc(&tm_tv);
    }
    for (int k = 0; k < BAR_COUNT; ++k) mbar_init(bar(k), (k == BAR_P_FULL || k == BAR_P_FULL + 1 || k == BAR_Q8) ? 4 : 1);
    *sT = 0;
    *sTailPos = -1;
    mbar_fence_init();
    fence_proxy_async();
  }
  if (warp == 5) {
    tmem_alloc(smem_u32(tmem_slot), kTmemCols);
    tmem_relinquish();
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");     // sel_idx / sel_cnt come from li_block_select (PDL)
  const int cnt = p.sel_cnt[row_id];
  const int32_t *sel_row = p.sel_idx + row_id * p.kmax;
  const int n_tiles = Nt + Nc + cnt;                   // attended tiles: text | chunk | selected history
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
  // ---- attended tile j (chunk blocks first, then the selected historical blocks) ----
  // 1-D: only two tiles can be partial: the last chunk block, and the history tail block M-1, wherever it sits in the
  // row's list (a row is a set: any order, li.h).  3-D: tiles of a region's last temporal group may hold fewer than bt
  // frames, border tiles fewer than bh grid rows.
  if (!k3d && tail_hist < BLK && cnt > 0) {            // CTA-uniform condition
    for (int t = threadIdx.x; t < cnt; t += blockDim.x)
      if (sel_at(t) == M - 1) *sTailPos = t;
    __syncthreads();
  }
  const int j_tail_hist = *sTailPos >= 0 ? Nt + Nc + *sTailPos : -1;
  auto tile_valid = [&](int j) -> int {                // 1-D tiles (and text tiles in both modes): valid prefix
    if (TEXT && j < Nt) return j == Nt - 1 ? tail_text : BLK;
    return j == Nt + Nc - 1 ? tail_cur : (j == j_tail_hist ? tail_hist : BLK);
  };
  auto tile_blk = [&](int j) -> int { return j < Nt + Nc ? j - Nt : sel_at(j - Nt - Nc); };   // block index in its region
  // 3-D: (frames of tile j that exist) | (valid grid columns if the block sticks out of the grid's right border, else 0) << 3
  //       | (grid rows inside the grid * bw = valid prefix of a full-width slice) << 8
  auto tile_info = [&](int j) -> int {
    int tg, hb, wb;
    split3(tile_blk(j), tg, hb, wb);
    const int nf = min(tl.bt, (j < Nt + Nc ? p.n_cur : n_hist) - tg * tl.bt);
    const int vw = tl.gw - wb * tl.bw;
    return nf | (vw < tl.bw ? vw : 0) << 3 | (min(tl.bh, tl.gh - hb * tl.bh) * tl.bw) << 8;
  };
  auto tile_info_cached = [&](int j) -> int { return j - Nt < kInfoCap ? (int)sInfo[j - Nt] : tile_info(j); };
  auto tile_frames = [&](int j) -> int { return tile_info_cached(j) & 7; };
  auto halves = [&](int j) -> int {                    // half-tiles of tile j with at least one valid key
    return (k3d && (!TEXT || j >= Nt)) ? (tile_frames(j) > SPH ? 2 : 1) : (tile_valid(j) > HALF ? 2 : 1);
  };
  // number of half-tiles with at least one valid key (a half-tile without any is skipped by every role)
  int T = 2 * n_tiles;
  if (k3d) {
    int part = 0;
    for (int j = threadIdx.x; j < n_tiles; j += blockDim.x) {
      if (TEXT && j < Nt) { part += tile_valid(j) > HALF ? 2 : 1; continue; }
      const int info = tile_info(j);                   // integer divisions once per tile, not once per half-tile per role
      if (j - Nt < kInfoCap) sInfo[j - Nt] = (uint16_t)info;
      part += (info & 7) > SPH ? 2 : 1;
    }
    if (part) atomicAdd(sT, part);
    __syncthreads();
    T = *sT;
  } else {
    if (TEXT && Nt > 0 && tail_text <= HALF) --T;
    if (Nc > 0 && tail_cur <= HALF) --T;
    if (j_tail_hist >= 0 && tail_hist <= HALF) --T;
  }

  // this CTA's range of half-tiles [t_lo, t_lo + Tn) (the whole list unless the query block is split)
  const int t_lo = (SPLIT && ns > 1) ? (int)((int64_t)T * sq / ns) : 0;
  const int Tn = (SPLIT && ns > 1) ? (int)((int64_t)T * (sq + 1) / ns) - t_lo : T;

  if (Tn > 0) {
    if (warp == 4) {
      // =============================== TMA producer ===============================
      // The warp stays converged (index arithmetic on warp-uniform values); an elected lane issues the TMA.
      if (elect_one()) {
        mbar_arrive_expect_tx(bar(BAR_Q_FULL), BLK * D * 2);
#pragma unroll
        for (int c = 0; c < D / 64; ++c) {
          if (k3d) {
            // query block i = (tg, hb, wb): one 32-row box per frame; a frame past the chunk is out of bounds -> zeros
            int tg, hb, wb;
            split3(i, tg, hb, wb);
            for (int tt = 0; tt < BLK / 32; ++tt)
              tma_load_5d(sQ + c * L::kQChunk + tt * 4096, &tm_q, bar(BAR_Q_FULL), c * 64, wb * tl.bw, hb * tl.bh,
                          min(tg * tl.bt + tt, n_qf), b * p.H + h);
          } else {
            tma_load_4d(sQ + c * L::kQChunk, &tm_q, bar(BAR_Q_FULL), c * 64, i * BLK, h, b);
          }
        }
      }
      __syncwarp();
      // the producer splits a block index twice per half-tile: multiply-high instead of two integer divisions
      const uint32_t mg_per = k3d ? 0xffffffffu / (uint32_t)max(per, 1) + 1u : 0u;   // (a divisor of 1 wraps to 0:
      const uint32_t mg_wb = k3d ? 0xffffffffu / (uint32_t)max(tl.Wb, 1) + 1u : 0u;  //  handled in split3_fast)
      auto split3_fast = [&](int blk, int &tg, int &hb, int &wb) {
        tg = per > 1 ? div_magic(blk, per, mg_per) : blk;
        const int r = blk - tg * per;
        hb = tl.Wb > 1 ? div_magic(r, tl.Wb, mg_wb) : r;
        wb = r - hb * tl.Wb;
      };
      int n = 0;                                     // running load index: slot = n % 4
      // loads HALF rows [t0, t0+HALF) of a region (history or chunk) into ring slot n % 4
      auto load_half = [&](const CUtensorMap *tm_full, const CUtensorMap *tm_8, const CUtensorMap *tm_text, int j, int hh) {
        const bool is_cur = j < Nt + Nc;
        const int blk = tile_blk(j);
        const int f0 = is_cur ? n_hist : 0;            // first frame of the region inside this call's frame list
        const int slot = n & (kStages - 1);
        const uint32_t dst = sRing + slot * L::kStage, mb = bar(BAR_FULL + slot);
        if (TEXT && j < Nt) {
          // text tile (T of Eq. 11): dense [B,H,Lt,d] tensor, rows past Lt are zero-filled by the hardware
          mbar_wait(bar(BAR_EMPTY + slot), ((n >> 2) & 1) ^ 1);
          if (elect_one()) {
            mbar_arrive_expect_tx(mb, HALF * D * 2);
#pragma unroll
            for (int c = 0; c < D / 64; ++c) tma_load_4d(dst + c * L::kKVChunk, tm_text, mb, c * 64, j * BLK + hh * HALF, h, b);   // text: bf16 only
          }
          __syncwarp();
          ++n;
          return;
        }
        if (k3d) {
          // 3-D block (tg, hb, wb): the half-tile is SPH frame slices of 32 rows (bh grid rows x bw columns), each one
          // 5-D box (64 channels, bw, bh, head, page); grid rows >= grid_h are zero-filled by the hardware ("masked
          // loads"); a frame past the region's end is requested out of bounds -> zeros
          const int n_reg = is_cur ? p.n_cur : n_hist;
          int tg, hb, wb;
          split3_fast(blk, tg, hb, wb);
          int pg[SPH], y0[SPH];
#pragma unroll
          for (int s = 0; s < SPH; ++s) {
            const int f = tg * tl.bt + hh * SPH + s;
            pg[s] = f < n_reg ? page_at(f0 + f) : 0;
            y0[s] = f < n_reg ? hb * tl.bh : tl.gh;
          }
          mbar_wait(bar(BAR_EMPTY + slot), ((n >> 2) & 1) ^ 1);
          if (elect_one()) {
            mbar_arrive_expect_tx(mb, HALF * D * EB);
#pragma unroll
            for (int s = 0; s < SPH; ++s)
#pragma unroll
              for (int c = 0; c < KCH; ++c)
                tma_load_5d(dst + c * L::kKVChunk + s * 4096, tm_full, mb, c * CW, wb * tl.bw, y0[s], h, pg[s]);
          }
          __syncwarp();
          ++n;
          return;
        }
        const int region_len = is_cur ? L_cur : L_hist;
        const int t0 = blk * BLK + hh * HALF;
        const int t_last = min(t0 + HALF, region_len) - 1;
        const int pg0 = t0 / p.T_f;
        const bool one_page = p.has_box_full && pg0 == t_last / p.T_f;
        const int page0 = page_at(f0 + pg0);
        mbar_wait(bar(BAR_EMPTY + slot), ((n >> 2) & 1) ^ 1);
        if (elect_one()) {
          mbar_arrive_expect_tx(mb, HALF * D * EB);
          if (one_page) {
            // inside one page: one box per 128-byte chunk; rows past the page end are zero-filled by the
            // hardware (a region always ends on a page boundary)
            const int row = t0 - pg0 * p.T_f;
#pragma unroll
            for (int c = 0; c < KCH; ++c) tma_load_4d(dst + c * L::kKVChunk, tm_full, mb, c * CW, row, h, page0);
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
              for (int c = 0; c < KCH; ++c)
                tma_load_4d(dst + c * L::kKVChunk + g * 1024, tm_8, mb, c * CW, row, h, page);
            }
          }
        }
        __syncwarp();
        ++n;
      };
      auto advance = [&](int &j, int &hh) {
        if (hh == 0 && halves(j) > 1) hh = 1;
        else { ++j; hh = 0; }
      };

      // load order == consumption order of the MMA warp: K0 K1 | V0 K2 | V1 K3 | ...
      int kj = 0, kh = 0, vj = 0, vh = 0;
      if (SPLIT) {                                   // split query block: skip to this CTA's range
        for (int t = 0; t < t_lo; ++t) advance(kj, kh);
        vj = kj; vh = kh;
      }
      load_half(&tm_k_full, &tm_k_8, &tm_tk, kj, kh); advance(kj, kh);
      if (Tn > 1) { load_half(&tm_k_full, &tm_k_8, &tm_tk, kj, kh); advance(kj, kh); }
      for (int t = 0; t < Tn; ++t) {
        load_half(&tm_v_full, &tm_v_8, &tm_tv, vj, vh); advance(vj, vh);
        if (t + 2 < Tn) { load_half(&tm_k_full, &tm_k_8, &tm_tk, kj, kh); advance(kj, kh); }
      }
    } else if (warp == 5) {
      // =============================== MMA issuer ===============================
      // The whole warp walks the loop converged (barrier waits, descriptor arithmetic on warp-uniform values);
      // one elected lane issues the tcgen05 instructions.
      constexpr uint32_t idesc_qk = KV8 ? idesc_e4m3(128, HALF, 0) : idesc_bf16(128, HALF, 0);
      constexpr uint32_t idesc_pv = KV8 ? idesc_e4m3(128, D, 1) : idesc_bf16(128, D, 1);
      const uint32_t sQ8 = smem_base + L::kOffQ8;
      int c = 0;                                     // running consume index: slot = c % 4
      auto issue_qk = [&](int t) {
        const int slot = c & (kStages - 1);
        const uint32_t sK = sRing + slot * L::kStage;
        mbar_wait(bar(BAR_FULL + slot), (c >> 2) & 1);
        tc_fence_after();
        if (elect_one()) {
          // descriptors of the kk-th 16-channel slice: the start address (16-byte units, cannot carry out of its
          // field) advances by 32 B inside the 128-B row and by one 64-channel chunk every 4 slices
          const uint64_t da0 = smem_desc_sw128(KV8 ? sQ8 : sQ, 16, 1024), db0 = smem_desc_sw128(sK, 16, 1024);
          if constexpr (KV8) {
            // e4m3: a 128-byte row holds all 128 channels; K = 32 channels = 32 bytes per instruction
#pragma unroll
            for (int kk = 0; kk < D / 32; ++kk)
              mma_ss_f8(tmem + (t & 1) * kSbCol, da0 + (uint64_t)((kk * 32) >> 4), db0 + (uint64_t)((kk * 32) >> 4), idesc_qk, kk > 0);
          } else {
#pragma unroll
            for (int kk = 0; kk < D / 16; ++kk)
              mma_ss(tmem + (t & 1) * kSbCol, da0 + (uint64_t)(((kk >> 2) * L::kQChunk + (kk & 3) * 32) >> 4),
                     db0 + (uint64_t)(((kk >> 2) * L::kKVChunk + (kk & 3) * 32) >> 4), idesc_qk, kk > 0);
          }
          mma_commit(bar(BAR_EMPTY + slot));
          mma_commit(bar(BAR_S_FULL + (t & 1)));
        }
        __syncwarp();
        ++c;
      };
      mbar_wait(bar(KV8 ? BAR_Q8 : BAR_Q_FULL), 0);
      issue_qk(0);
      if (Tn > 1) issue_qk(1);
      for (int t = 0; t < Tn; ++t) {
        // O += P(t) V(t)
        const int slot = c & (kStages - 1);
        const uint32_t sV = sRing + slot * L::kStage;
        mbar_wait(bar(BAR_FULL + slot), (c >> 2) & 1);
        mbar_wait(bar(BAR_P_FULL + (t & 1)), (t >> 1) & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t db0 = smem_desc_sw128(sV, L::kKVChunk, 1024);
          if constexpr (KV8) {
            // P in e4m3: 32 keys = 8 TMEM columns per instruction; V rows (keys) of 128 bytes = all d channels, 32 rows on
#pragma unroll
            for (int kk = 0; kk < HALF / 32; ++kk)
              mma_ts_f8(tmem + kOCol, tmem + (t & 1) * kSbCol + kk * 8, db0 + (uint64_t)((kk * 4096) >> 4), idesc_pv,
                        (t > 0 || kk > 0) ? 1u : 0u);
          } else {
#pragma unroll
            for (int kk = 0; kk < HALF / 16; ++kk)
              mma_ts(tmem + kOCol, tmem + (t & 1) * kSbCol + kk * 8, db0 + (uint64_t)((kk * 2048) >> 4), idesc_pv,
                     (t > 0 || kk > 0) ? 1u : 0u);
          }
          mma_commit(bar(BAR_EMPTY + slot));
          mma_commit(bar(BAR_PV_DONE));
          if (t == Tn - 1) mma_commit(bar(BAR_O_FULL));
        }
        __syncwarp();
        ++c;
        if (t + 2 < Tn) issue_qk(t + 2);
      }
    } else {
      // =============================== softmax / lazy correction / epilogue ===============================
      const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
      const int row = warp * 32 + lane;                // query row inside the tile == TMEM lane
      float m_used = 0.f, l = 0.f;
      float scale_row = p.scale_log2;                  // logits (log2 units) per unit of the raw dot product S
      if constexpr (KV8) {
        // FP8 pages: both MMA operands are 8-bit, so the query row of this thread is replaced by its own e4m3 image:
        // qs = max|q| / 448 (fp32; 1 for a zero row), code = e4m3(q / qs).  The bf16 row is read from the TMA-written
        // tile (SWIZZLE_128B: 16-byte piece j of row r sits at piece j ^ (r mod 8)) and the codes are written in the
        // same K-major swizzled layout, one 128-byte row per query.
        mbar_wait(bar(BAR_Q_FULL), 0);
        const uint8_t *qrow = smem + L::kOffQ + (row >> 3) * 1024 + (row & 7) * 128;
        float amax = 0.f;
#pragma unroll
        for (int c = 0; c < D / 64; ++c)
#pragma unroll
          for (int jp = 0; jp < 8; ++jp) {
            const uint4 v = *reinterpret_cast<const uint4 *>(qrow + c * L::kQChunk + ((jp ^ (row & 7)) << 4));
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int e = 0; e < 4; ++e)
              amax = fmaxf(amax, fmaxf(fabsf(__uint_as_float(w[e] << 16)), fabsf(__uint_as_float(w[e] & 0xffff0000u))));
          }
        const float qs = amax > 0.f ? __fdiv_rn(amax, 448.0f) : 1.0f;
        uint8_t *q8row = smem + L::kOffQ8 + (row >> 3) * 1024 + (row & 7) * 128;
#pragma unroll
        for (int jo = 0; jo < 8; ++jo) {               // output piece jo = channels 16 jo .. 16 jo + 15 = two bf16 pieces
          uint32_t out[4];
#pragma unroll
          for (int half_ = 0; half_ < 2; ++half_) {
            const int ch = jo * 16 + half_ * 8, c = ch >> 6, jp = (ch & 63) >> 3;
            const uint4 v = *reinterpret_cast<const uint4 *>(qrow + c * L::kQChunk + ((jp ^ (row & 7)) << 4));
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              const float x0 = __fdiv_rn(__uint_as_float(w[2 * e] << 16), qs), x1 = __fdiv_rn(__uint_as_float(w[2 * e] & 0xffff0000u), qs);
              const float x2 = __fdiv_rn(__uint_as_float(w[2 * e + 1] << 16), qs), x3 = __fdiv_rn(__uint_as_float(w[2 * e + 1] & 0xffff0000u), qs);
              out[half_ * 2 + e] = pack_e4m3x2(x0, x1) | (pack_e4m3x2(x2, x3) << 16);
            }
          }
          *reinterpret_cast<uint4 *>(q8row + ((jo ^ (row & 7)) << 4)) = make_uint4(out[0], out[1], out[2], out[3]);
        }
        fence_proxy_async();                           // generic-proxy writes -> visible to the tensor core's smem reads
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_Q8));
        scale_row = p.scale_log2 * qs * __ldg(p.k_scale + h);   // S = (q / qs) . (k / ks): logits = S * qs * ks * scale
      }
      int j = 0, hh = 0;
      if (SPLIT) {                                     // split query block: skip to this CTA's range
        for (int t = 0; t < t_lo; ++t) {
          if (hh == 0 && halves(j) > 1) hh = 1;
          else { ++j; hh = 0; }
        }
      }

      for (int t = 0; t < Tn; ++t) {
        // valid key columns of this half-tile, as a prefix length per 32-column slice (vs[s] keys of slice s are real, the
        // rest is padding): 1-D blocks have one valid prefix; a 3-D slice is one frame's bh x bw patch (key (y, x) in
        // column y * bw + x), whose grid rows beyond grid_h (and whose frame, beyond the region) are padding; in a block
        // over the grid's right border only vw of the bw columns exist
        int vs[SPH];
        int vw = 0;
        if (k3d && (!TEXT || j >= Nt)) {
          const int info = tile_info_cached(j), nf = info & 7, vrow = info >> 8;
          vw = (info >> 3) & 31;
#pragma unroll
          for (int s_ = 0; s_ < SPH; ++s_) vs[s_] = (hh * SPH + s_ < nf) ? vrow : 0;
        } else {
          const int hv = min(HALF, tile_valid(j) - hh * HALF);
#pragma unroll
          for (int s_ = 0; s_ < SPH; ++s_) vs[s_] = min(32, max(0, hv - 32 * s_));
        }
        bool rows_full = true;
#pragma unroll
        for (int s_ = 0; s_ < SPH; ++s_) rows_full = rows_full && vs[s_] == 32;
        if (hh == 0 && halves(j) > 1) hh = 1;
        else { ++j; hh = 0; }
        const uint32_t s_addr = tmem + lane_base + (t & 1) * kSbCol;

        mbar_wait(bar(BAR_S_FULL + (t & 1)), (t >> 1) & 1);
        tc_fence_after();
        uint32_t s[HALF];
#pragma unroll
        for (int c = 0; c < HALF / 32; ++c) tmem_ld32(s_addr + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&s[c * 32]));
        tc_wait_ld();
        if (!rows_full) {                              // padded key rows -> -inf (warp-uniform branch)
          bool same = k3d;                               // 3-D border tile: every slice has the same valid prefix,
#pragma unroll
          for (int s_ = 1; s_ < SPH; ++s_) same = same && vs[s_] == vs[0];   // a multiple of bw rows
          if (same && (vs[0] & 7) == 0 && vs[0] > 0) {
            // compile-time column positions: a few moves, no compares
            if (vs[0] == 24) mask_slice_tail<24, HALF>(s);
            else if (vs[0] == 16) mask_slice_tail<16, HALF>(s);
            else mask_slice_tail<8, HALF>(s);
          } else {
#pragma unroll
            for (int c = 0; c < HALF; ++c) if ((c & 31) >= vs[c >> 5]) s[c] = 0xff800000u;
          }
        }
        if (k3d && vw != 0) {                          // right-border block: grid columns x >= vw lie outside the grid
          const int xm = tl.bw - 1;
#pragma unroll
          for (int c = 0; c < HALF; ++c) if ((c & xm) >= vw) s[c] = 0xff800000u;
        }
        float mx0 = __uint_as_float(s[0]), mx1 = __uint_as_float(s[1]), mx2 = __uint_as_float(s[2]), mx3 = __uint_as_float(s[3]);
#pragma unroll
        for (int c = 4; c < HALF; c += 4) {
          mx0 = fmaxf(mx0, __uint_as_float(s[c]));
          mx1 = fmaxf(mx1, __uint_as_float(s[c + 1]));
          mx2 = fmaxf(mx2, __uint_as_float(s[c + 2]));
          mx3 = fmaxf(mx3, __uint_as_float(s[c + 3]));
        }
        const float m_new = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * scale_row;

        // lazy rescale: the reference maximum only moves when the row maximum grew by more than 2^8
        bool need = false;
        if (t == 0) m_used = m_new;
        else need = m_new > m_used + kRescaleThreshold;
        if (__ballot_sync(0xffffffffu, need)) {
          // O is being accumulated by PV(t-1): wait for it (PV(t-2) is known complete, so the parity is unambiguous)
          mbar_wait(bar(BAR_PV_DONE), (t - 1) & 1);
          tc_fence_after();
          const float f = need ? ex2_approx(m_used - m_new) : 1.0f;
          if (need) { m_used = m_new; l *= f; }
#pragma unroll 1
          for (int c = 0; c < D / 32; ++c) {
            uint32_t o[32];
            tmem_ld32(tmem + lane_base + kOCol + c * 32, o);
            tc_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * f);
            tmem_st32(tmem + lane_base + kOCol + c * 32, o);
          }
        }

        // P = exp2(s*scale - m_used), row sum in fp32, bf16 pairs packed low = even column.  kEmuOf4 of every 4
        // column pairs take the FMA-pipe exp2 (li_ptx.cuh), the others the MUFU, so that both pipes stay busy.
        const uint64_t sc2 = pack2(scale_row, scale_row), nm2 = pack2(-m_used, -m_used);
        uint64_t sum_a = pack2(0.f, 0.f), sum_b = pack2(0.f, 0.f);
        uint32_t pk[HALF / 2];
#pragma unroll
        for (int c = 0; c < HALF / 2; ++c) {
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
          if constexpr (KV8) {                           // e4m3: four keys per 32-bit TMEM column, lowest key in the low byte
            if (c & 1) pk[c >> 1] |= pack_e4m3x2(p0, p1) << 16;
            else pk[c >> 1] = pack_e4m3x2(p0, p1);
          } else {
            pk[c] = pack_bf16x2(p0, p1);
          }
        }
        {
          float a0, a1;
          unpack2(add2(sum_a, sum_b), a0, a1);
          l += a0 + a1;
        }
        if constexpr (KV8) tmem_st16(s_addr, pk);      // 64 keys in e4m3 = 16 columns (FP8 pages: BLK == 128)
        else if constexpr (HALF == 64) tmem_st32(s_addr, *reinterpret_cast<uint32_t(*)[32]>(&pk[0]));
        else tmem_st16(s_addr, pk);
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_P_FULL + (t & 1)));
      }


      mbar_wait(bar(BAR_O_FULL), 0);
      tc_fence_after();
      if (SPLIT && ns > 1) {
        // split query block: unnormalised fp32 partial O and (reference maximum, row sum) for li_attn_combine_kernel
        const int64_t prow = (int64_t)(blockIdx.x - p.split_first) * 128 + row;
        float *po = p.part_o + prow * D;
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
          uint32_t o[32];
          tmem_ld32(tmem + lane_base + kOCol + c * 32, o);
          tc_wait_ld();
          if constexpr (KV8) {                           // O accumulates P . (v / vs): the per-head V scale goes in here
            const float vs = __ldg(p.v_scale + h);
#pragma unroll
            for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * vs);
          }
#pragma unroll
          for (int e = 0; e < 32; e += 4)
            *reinterpret_cast<uint4 *>(po + c * 32 + e) = make_uint4(o[e], o[e + 1], o[e + 2], o[e + 3]);
        }
        p.part_ml[prow] = make_float2(m_used, l);
      } else {
        // epilogue: O / l -> bf16, stored in linear token order (no untile pass)
        const float inv_l = (KV8 ? __ldg(p.v_scale + h) : 1.0f) / l;   // FP8 pages: O accumulated P . (v / vs)
        const int64_t u = row_token<BLK, K3D>(p, i, row);
        const bool live = u >= 0;
        uint16_t *orow = p.o + (((int64_t)b * p.H + h) * p.Lq + u) * D;
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
          uint32_t o[32];
          tmem_ld32(tmem + lane_base + kOCol + c * 32, o);
          tc_wait_ld();
          if (live) {
#pragma unroll
            for (int e = 0; e < 32; e += 8) {
              uint4 v;
              v.x = pack_bf16x2(__uint_as_float(o[e + 0]) * inv_l, __uint_as_float(o[e + 1]) * inv_l);
              v.y = pack_bf16x2(__uint_as_float(o[e + 2]) * inv_l, __uint_as_float(o[e + 3]) * inv_l);
              v.z = pack_bf16x2(__uint_as_float(o[e + 4]) * inv_l, __uint_as_float(o[e + 5]) * inv_l);
              v.w = pack_bf16x2(__uint_as_float(o[e + 6]) * inv_l, __uint_as_float(o[e + 7]) * inv_l);
              *reinterpret_cast<uint4 *>(orow + c * 32 + e) = v;
            }
          }
        }
        if (live && p.lse != nullptr)
          p.lse[((int64_t)b * p.H + h) * p.Lq + u] = (m_used + log2f(l)) * 0.6931471805599453f;
      }
    }
  } else {
    // no half-tile for this CTA (empty context, or a split range without tiles)
    if (warp < 4) {
      const int row = warp * 32 + lane;
      if (SPLIT && ns > 1) {
        p.part_ml[(int64_t)(blockIdx.x - p.split_first) * 128 + row] = make_float2(0.f, 0.f);   // row sum 0: ignored
      } else {
        const int64_t u = row_token<BLK, K3D>(p, i, row);   // o = 0, lse = -inf
        if (u >= 0) {
          uint16_t *orow = p.o + (((int64_t)b * p.H + h) * p.Lq + u) * D;
          for (int c = 0; c < D; c += 8) *reinterpret_cast<uint4 *>(orow + c) = make_uint4(0, 0, 0, 0);
          if (p.lse != nullptr) p.lse[((int64_t)b * p.H + h) * p.Lq + u] = __int_as_float(0xff800000);
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 5) tmem_dealloc(tmem, kTmemCols);
}

// Two entry points: the text maps are kernel parameters only of the variant that attends a text prefix (adding two
// unused 128-byte tensor maps to the parameter block of the plain kernel measurably slowed it down).
template <int D, int BLK, bool K3D, bool SPLIT>
__global__ void __launch_bounds__(192, 2)
li_sparse_attn_kernel(const AttnParams p, const BatchMeta meta, const __grid_constant__ CUtensorMap tm_q,
                      const __grid_constant__ CUtensorMap tm_k_full, const __grid_constant__ CUtensorMap tm_k_8,
                      const __grid_constant__ CUtensorMap tm_v_full, const __grid_constant__ CUtensorMap tm_v_8) {
  attn_body<D, BLK, K3D, false, SPLIT, false>(p, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8, tm_q, tm_q);
}

// FP8 (E4M3) K/V pages: both contractions on the kind::f8f6f4 tensor-core path (d = 128, 128-token blocks)
template <bool K3D, bool SPLIT>
__global__ void __launch_bounds__(192, 2)
li_sparse_attn_fp8_kernel(const AttnParams p, const BatchMeta meta, const __grid_constant__ CUtensorMap tm_q,
                          const __grid_constant__ CUtensorMap tm_k_full, const __grid_constant__ CUtensorMap tm_k_8,
                          const __grid_constant__ CUtensorMap tm_v_full, const __grid_constant__ CUtensorMap tm_v_8) {
  attn_body<128, 128, K3D, false, SPLIT, true>(p, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8, tm_q, tm_q);
}

template <int D, int BLK, bool K3D, bool SPLIT>
__global__ void __launch_bounds__(192, 2)
li_sparse_attn_text_kernel(const AttnParams p, const BatchMeta meta, const __grid_constant__ CUtensorMap tm_q,
                           const __grid_constant__ CUtensorMap tm_k_full, const __grid_constant__ CUtensorMap tm_k_8,
                           const __grid_constant__ CUtensorMap tm_v_full, const __grid_constant__ CUtensorMap tm_v_8,
                           const __grid_constant__ CUtensorMap tm_tk, const __grid_constant__ CUtensorMap tm_tv) {
  attn_body<D, BLK, K3D, true, SPLIT, false>(p, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8, tm_tk, tm_tv);
}

// Merges the n_split partial results of every split query block (tail-wave split): with reference maxima
// m_q and row sums l_q, O = sum_q 2^(m_q - M) O_q / sum_q 2^(m_q - M) l_q, M = max_q m_q over the parts that saw a key.
// grid (split query blocks, 16), 8 warps: one warp per query row, lane = D/32 consecutive channels.
template <int D, int BLK, bool K3D>
__global__ void __launch_bounds__(256) li_attn_combine_kernel(const AttnParams p) {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int work = p.split_first + blockIdx.x, row = blockIdx.y * 8 + warp;
  const int i = work % p.Nqb, h = (work / p.Nqb) % p.H, b = work / (p.Nqb * p.H);
  const int64_t u = row_token<BLK, K3D>(p, i, row);
  if (u < 0) return;
  constexpr int V = D / 32;
  const int64_t prow0 = (int64_t)blockIdx.x * p.n_split * 128 + row;
  float M = __int_as_float(0xff800000);
  for (int q = 0; q < p.n_split; ++q) {
    const float2 ml = p.part_ml[prow0 + (int64_t)q * 128];
    if (ml.y > 0.f) M = fmaxf(M, ml.x);
  }
  float L = 0.f, acc[V];
#pragma unroll
  for (int c = 0; c < V; ++c) acc[c] = 0.f;
  for (int q = 0; q < p.n_split; ++q) {
    const float2 ml = p.part_ml[prow0 + (int64_t)q * 128];
    if (ml.y > 0.f) {
      const float w = exp2f(ml.x - M);
      L += w * ml.y;
      const float *po = p.part_o + (prow0 + (int64_t)q * 128) * D + lane * V;
#pragma unroll
      for (int c = 0; c < V; ++c) acc[c] += w * po[c];
    }
  }
  const float inv = L > 0.f ? 1.0f / L : 0.f;
  uint16_t *orow = p.o + (((int64_t)b * p.H + h) * p.Lq + u) * D + lane * V;
#pragma unroll
  for (int c = 0; c < V; c += 2) *reinterpret_cast<uint32_t *>(orow + c) = pack_bf16x2(acc[c] * inv, acc[c + 1] * inv);
  if (lane == 0 && p.lse != nullptr)
    p.lse[((int64_t)b * p.H + h) * p.Lq + u] = L > 0.f ? (M + log2f(L)) * 0.6931471805599453f : __int_as_float(0xff800000);
}

template <int D, int BLK, bool K3D, bool TEXT, bool SPLIT, bool KV8 = false>
static int launch_one(const AttnParams &ap, const BatchMeta &meta, const CUtensorMap &tm_q, const CUtensorMap &tm_tk,
                      const CUtensorMap &tm_tv, const CUtensorMap &tm_k_full,
                      const CUtensorMap &tm_k_8, const CUtensorMap &tm_v_full, const CUtensorMap &tm_v_8,
                      cudaStream_t st) {
  constexpr int smem = AttnSmem<D, BLK, KV8>::kTotal;
  cudaError_t e;
  // the dynamic shared-memory limit of this instance is raised once per device, not on every call
  static std::atomic<uint64_t> attr_done{0};
  int dev = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return (int)e;
  const uint64_t dev_bit = 1ull << (dev & 63);
  if (!(attr_done.load(std::memory_order_acquire) & dev_bit)) {
    if constexpr (KV8) e = cudaFuncSetAttribute(li_sparse_attn_fp8_kernel<K3D, SPLIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    else if constexpr (TEXT) e = cudaFuncSetAttribute(li_sparse_attn_text_kernel<D, BLK, K3D, SPLIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    else e = cudaFuncSetAttribute(li_sparse_attn_kernel<D, BLK, K3D, SPLIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return (int)e;
    attr_done.fetch_or(dev_bit, std::memory_order_release);
  }
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  const int n_work = ap.Nqb * ap.H * ap.B;
  cfg.gridDim = SPLIT ? dim3(ap.split_first + (n_work - ap.split_first) * ap.n_split) : dim3(ap.Nqb, ap.H, ap.B);
  cfg.blockDim = dim3(192);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if constexpr (KV8)
    e = cudaLaunchKernelEx(&cfg, li_sparse_attn_fp8_kernel<K3D, SPLIT>, ap, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8);
  else if constexpr (TEXT)
    e = cudaLaunchKernelEx(&cfg, li_sparse_attn_text_kernel<D, BLK, K3D, SPLIT>, ap, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8, tm_tk, tm_tv);
  else
    e = cudaLaunchKernelEx(&cfg, li_sparse_attn_kernel<D, BLK, K3D, SPLIT>, ap, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8);
  if (e != cudaSuccess) return (int)e;
  if (SPLIT) {
    cfg.gridDim = dim3(n_work - ap.split_first, 16);
    cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = 0;
    e = cudaLaunchKernelEx(&cfg, li_attn_combine_kernel<D, BLK, K3D>, ap);
    if (e != cudaSuccess) return (int)e;
  }
  return (int)cudaGetLastError();
}

int launch_attn(const AttnParams &ap_in, const BatchMeta &meta, int d, int blk, const CUtensorMap &tm_q,
                const CUtensorMap &tm_tk, const CUtensorMap &tm_tv, const CUtensorMap &tm_k_full, const CUtensorMap &tm_k_8, const CUtensorMap &tm_v_full,
                const CUtensorMap &tm_v_8, cudaStream_t st, int64_t *n_launches) {
  int e;
  AttnParams ap = ap_in;
  const bool k3 = ap.tl.bt > 0;
  // Tail-wave split.  The GPU holds `slots` = 2 CTAs per SM at a time; when the last wave would fill at
  // most half of them, its `rem` query blocks are each shared by s CTAs (s * rem <= slots), so the tail takes ~1/s of
  // a wave.  Needs the partial-result buffers (caller passed a full-size workspace); LI_FLAG_NO_SPLIT turns it off.
  const int n_work = ap.Nqb * ap.H * ap.B;
  ap.split_first = n_work;
  ap.n_split = 1;
  const int n_sm = (ap.part_o != nullptr && !ap.no_split) ? device_sm_count() : 0;
  if (n_sm > 0) {
    const int wave = 2 * n_sm, slots = wave < kMaxSplitSlots ? wave : kMaxSplitSlots;
    const int rem = n_work % wave;
    if (rem > 0 && 2 * rem <= slots) {
      const int t_est = 2 * ((ap.Lt + blk - 1) / blk + ap.Nc + ap.kmax);   // half-tiles per query block, upper bound
      int s = slots / rem;
      if (s > 8) s = 8;
      // at least ~16 half-tiles per CTA in a tail wave; a grid that fills less than one wave is pure latency, there 6
      // half-tiles per CTA still pay for the merge (`tiny`: 26.2 -> 18.0 us, thresholds 16 / 8 / 6 / 4 measured)
      const int min_ht = n_work < wave ? 6 : 16;
      if (s > t_est / min_ht) s = t_est / min_ht;
      if (s >= 2) {
        ap.n_split = s;
        ap.split_first = n_work - rem;
      }
    }
  }
#define LI_LAUNCH3(DD, BB, K3, TX)                                                                                    \
  (ap.n_split > 1 ? launch_one<DD, BB, K3, TX, true>(ap, meta, tm_q, tm_tk, tm_tv, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st) \
                  : launch_one<DD, BB, K3, TX, false>(ap, meta, tm_q, tm_tk, tm_tv, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st))
#define LI_LAUNCH2(DD, BB, K3) (ap.Lt > 0 ? LI_LAUNCH3(DD, BB, K3, true) : LI_LAUNCH3(DD, BB, K3, false))
#define LI_LAUNCH(DD, BB) (k3 ? LI_LAUNCH2(DD, BB, true) : LI_LAUNCH2(DD, BB, false))
#define LI_LAUNCH_FP8(K3) \
  (ap.n_split > 1 ? launch_one<128, 128, K3, false, true, true>(ap, meta, tm_q, tm_tk, tm_tv, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st) \
                  : launch_one<128, 128, K3, false, false, true>(ap, meta, tm_q, tm_tk, tm_tv, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st))
  if (ap.k_scale != nullptr) e = k3 ? LI_LAUNCH_FP8(true) : LI_LAUNCH_FP8(false);   // FP8 pages: d = 128, block 128 (checked by the API)
  else if (d == 128 && blk == 128) e = LI_LAUNCH(128, 128);
  else if (d == 128 && blk == 64) e = LI_LAUNCH(128, 64);
  else if (d == 64 && blk == 128) e = LI_LAUNCH(64, 128);
  else e = LI_LAUNCH(64, 64);
#undef LI_LAUNCH
#undef LI_LAUNCH_FP8
#undef LI_LAUNCH2
#undef LI_LAUNCH3
  if (e == 0 && n_launches) *n_launches += ap.n_split > 1 ? 2 : 1;
  return e;
}

}  // namespace li
