// li_attn.cu -- li_sparse_attn for sm_100a: block-sparse flash attention over C_i = K^curr U S_i
// (Eq. 11), K/V tiles fetched IN PLACE from the frame-paged cache by TMA with the page
// as a tensor coordinate (replaces the paper's KV-Prep / Untile-Scatter copies).
//
// One CTA = one query block (BLK query rows, padded to the 128-row UMMA tile) of one (call, head).
// Two CTAs are resident per SM (256 TMEM columns and ~98 KB of shared memory each), so that one CTA's
// softmax overlaps the other CTA's MMAs.
//   warps 0-3 : softmax + correction + epilogue; warp w owns TMEM lanes 32w..32w+31 (one query row per thread)
//   warp 4    : TMA producer (one elected lane): Q once, then K_j / V_j per attended block
//   warp 5    : TMEM allocation and the single-thread tcgen05.mma issuer
// TMEM: columns [0,BLK) S (fp32), overlaid by P (bf16, BLK/2 columns) once S has been read; [128,128+D) O.
#include "li_internal.h"
#include "li_ptx.cuh"

namespace li {

constexpr int kSelCap = 1024;       // selected-block indices staged in shared memory (rest read from global)
constexpr int kTmemCols = 256;
constexpr int kOCol = 128;
constexpr float kRescaleThreshold = 8.0f;   // log2 units: P stays <= 2^8 between lazy rescales

template <int D, int BLK>
struct AttnSmem {
  static constexpr int kQChunk = 128 * 128;            // bytes of one 64-column chunk of the 128-row Q tile
  static constexpr int kKVChunk = BLK * 128;           // bytes of one 64-column chunk of a K or V tile
  static constexpr int kQ = (D / 64) * kQChunk;
  static constexpr int kKV = (D / 64) * kKVChunk;
  static constexpr int kOffQ = 0;
  static constexpr int kOffK = kQ;
  static constexpr int kOffV = kQ + kKV;
  static constexpr int kOffSel = kQ + 2 * kKV;
  static constexpr int kOffBar = kOffSel + kSelCap * 4;
  static constexpr int kTotal = kOffBar + 128 + 1024;  // + barriers + slack for 1024-B alignment
};

enum { BAR_Q_FULL = 0, BAR_K_FULL, BAR_K_EMPTY, BAR_V_FULL, BAR_V_EMPTY, BAR_S_FULL, BAR_P_FULL, BAR_O_FULL, BAR_COUNT };

template <int D, int BLK>
__global__ void __launch_bounds__(192, 2)
li_sparse_attn_kernel(const AttnParams p, const BatchMeta meta, const __grid_constant__ CUtensorMap tm_q,
                      const __grid_constant__ CUtensorMap tm_k_full, const __grid_constant__ CUtensorMap tm_k_8,
                      const __grid_constant__ CUtensorMap tm_v_full, const __grid_constant__ CUtensorMap tm_v_8) {
  using L = AttnSmem<D, BLK>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *smem = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t sQ = smem_base + L::kOffQ, sK = smem_base + L::kOffK, sV = smem_base + L::kOffV;
  int32_t *sSel = reinterpret_cast<int32_t *>(smem + L::kOffSel);
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
  const int cnt = p.sel_cnt[row_id];
  const int32_t *sel_row = p.sel_idx + row_id * p.kmax;
  const int n_tiles = Nc + cnt;
  const int valid_q = min(BLK, p.Lq - i * BLK);

  // ---- one-time setup ----
  for (int t = threadIdx.x; t < cnt && t < kSelCap; t += blockDim.x) sSel[t] = sel_row[t];
  if (warp == 4 && lane == 0) {
    tma_prefetch_desc(&tm_q);
    tma_prefetch_desc(&tm_k_full);
    tma_prefetch_desc(&tm_v_full);
    tma_prefetch_desc(&tm_k_8);
    tma_prefetch_desc(&tm_v_8);
    for (int k = 0; k < BAR_COUNT; ++k) mbar_init(bar(k), k == BAR_P_FULL ? 4 : 1);
    mbar_fence_init();
    fence_proxy_async();
  }
  if (warp == 5) {
    tmem_alloc(smem_u32(tmem_slot), kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  auto sel_at = [&](int jj) -> int { return jj < kSelCap ? sSel[jj] : sel_row[jj]; };

  if (n_tiles > 0) {
    if (warp == 4) {
      // =============================== TMA producer ===============================
      if (lane == 0) {
        mbar_arrive_expect_tx(bar(BAR_Q_FULL), BLK * D * 2);
#pragma unroll
        for (int c = 0; c < D / 64; ++c) tma_load_4d(sQ + c * L::kQChunk, &tm_q, bar(BAR_Q_FULL), c * 64, i * BLK, h, b);

        auto issue_tile = [&](const CUtensorMap *tm_full, const CUtensorMap *tm_8, uint32_t dst, uint32_t mb,
                              const int32_t *pages, int t0, int region_len) {
          const int t_last = min(t0 + BLK, region_len) - 1;
          const int pg0 = t0 / p.T_f;
          if (p.has_box_full && pg0 == t_last / p.T_f) {
            // whole block inside one page: one box per 64-column chunk; rows past the page end are
            // zero-filled by the hardware (the region always ends on a page boundary)
            const int page = pages[pg0];
            const int row = t0 - pg0 * p.T_f;
#pragma unroll
            for (int c = 0; c < D / 64; ++c) tma_load_4d(dst + c * L::kKVChunk, tm_full, mb, c * 64, row, h, page);
          } else {
            // block straddles frames: 8-row pieces (one SWIZZLE_128B atom each, destinations stay 1024-B aligned)
            int cur_pg = -1, page = 0;
            for (int g = 0; g < BLK / 8; ++g) {
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
        };

        for (int j = 0; j < n_tiles; ++j) {
          const bool is_cur = j < Nc;
          const int blk = is_cur ? j : sel_at(j - Nc);
          const int32_t *pages = p.frame_idx + foff + (is_cur ? n_hist : 0);
          const int region_len = is_cur ? L_cur : L_hist;
          const uint32_t ph = (j & 1) ^ 1;
          mbar_wait(bar(BAR_K_EMPTY), ph);
          mbar_arrive_expect_tx(bar(BAR_K_FULL), BLK * D * 2);
          issue_tile(&tm_k_full, &tm_k_8, sK, bar(BAR_K_FULL), pages, blk * BLK, region_len);
          mbar_wait(bar(BAR_V_EMPTY), ph);
          mbar_arrive_expect_tx(bar(BAR_V_FULL), BLK * D * 2);
          issue_tile(&tm_v_full, &tm_v_8, sV, bar(BAR_V_FULL), pages, blk * BLK, region_len);
        }
      }
    } else if (warp == 5) {
      // =============================== MMA issuer ===============================
      if (lane == 0) {
        constexpr uint32_t idesc_qk = idesc_bf16(128, BLK, 0);
        constexpr uint32_t idesc_pv = idesc_bf16(128, D, 1);
        mbar_wait(bar(BAR_Q_FULL), 0);
        for (int j = 0; j < n_tiles; ++j) {
          const uint32_t ph = j & 1;
          // S = Q K^T
          mbar_wait(bar(BAR_K_FULL), ph);
          tc_fence_after();
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            const uint64_t da = smem_desc_sw128(sQ + (kk >> 2) * L::kQChunk + (kk & 3) * 32, 16, 1024);
            const uint64_t db = smem_desc_sw128(sK + (kk >> 2) * L::kKVChunk + (kk & 3) * 32, 16, 1024);
            mma_ss(tmem, da, db, idesc_qk, kk > 0);
          }
          mma_commit(bar(BAR_K_EMPTY));
          mma_commit(bar(BAR_S_FULL));
          // O += P V
          mbar_wait(bar(BAR_V_FULL), ph);
          mbar_wait(bar(BAR_P_FULL), ph);
          tc_fence_after();
#pragma unroll
          for (int kk = 0; kk < BLK / 16; ++kk) {
            const uint64_t db = smem_desc_sw128(sV + kk * 2048, L::kKVChunk, 1024);
            mma_ts(tmem + kOCol, tmem + kk * 8, db, idesc_pv, (j > 0 || kk > 0) ? 1u : 0u);
          }
          mma_commit(bar(BAR_V_EMPTY));
          if (j == n_tiles - 1) mma_commit(bar(BAR_O_FULL));
        }
      }
      __syncwarp();
    } else {
      // =============================== softmax / correction / epilogue ===============================
      const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
      const int row = warp * 32 + lane;                // query row inside the tile == TMEM lane
      float m_used = 0.f, l = 0.f;
      const int tail_cur = L_cur - (Nc - 1) * BLK, tail_hist = L_hist - (M - 1) * BLK;

      for (int j = 0; j < n_tiles; ++j) {
        int valid = BLK;
        if (j < Nc) { if (j == Nc - 1) valid = tail_cur; }
        else if (sel_at(j - Nc) == M - 1) valid = tail_hist;

        mbar_wait(bar(BAR_S_FULL), j & 1);
        tc_fence_after();
        uint32_t s[BLK];
#pragma unroll
        for (int c = 0; c < BLK / 32; ++c) tmem_ld32(tmem + lane_base + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&s[c * 32]));
        tc_wait_ld();
        if (valid < BLK) {                             // padded key columns -> -inf (warp-uniform branch)
#pragma unroll
          for (int c = 0; c < BLK; ++c) if (c >= valid) s[c] = 0xff800000u;
        }
        float mx = __uint_as_float(s[0]);
#pragma unroll
        for (int c = 1; c < BLK; ++c) mx = fmaxf(mx, __uint_as_float(s[c]));
        const float m_new = mx * p.scale_log2;

        // lazy rescale: move the reference maximum only when the row maximum grew by more than 2^8
        bool need = false;
        if (j == 0) m_used = m_new;
        else need = m_new > m_used + kRescaleThreshold;
        if (__ballot_sync(0xffffffffu, need)) {
          const float f = need ? ex2_approx(m_used - m_new) : 1.0f;
          if (need) { m_used = m_new; l *= f; }
#pragma unroll
          for (int c = 0; c < D / 32; ++c) {
            uint32_t o[32];
            tmem_ld32(tmem + lane_base + kOCol + c * 32, o);
            tc_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * f);
            tmem_st32(tmem + lane_base + kOCol + c * 32, o);
          }
        }

        // P = exp2(s*scale - m_used), row sum in fp32, bf16 pairs packed low = even column
        const float neg_m = -m_used;
        float sum0 = 0.f, sum1 = 0.f;
        uint32_t pk[BLK / 2];
#pragma unroll
        for (int c = 0; c < BLK / 2; ++c) {
          const float p0 = ex2_approx(fmaf(__uint_as_float(s[2 * c]), p.scale_log2, neg_m));
          const float p1 = ex2_approx(fmaf(__uint_as_float(s[2 * c + 1]), p.scale_log2, neg_m));
          sum0 += p0;
          sum1 += p1;
          pk[c] = pack_bf16x2(p0, p1);
        }
        l += sum0 + sum1;
#pragma unroll
        for (int c = 0; c < BLK / 64; ++c) tmem_st32(tmem + lane_base + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&pk[c * 32]));
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(BAR_P_FULL));
      }

      // epilogue: O / l -> bf16, stored in linear token order (no untile pass)
      mbar_wait(bar(BAR_O_FULL), 0);
      tc_fence_after();
      const float inv_l = 1.0f / l;
      const bool live = row < valid_q;
      uint16_t *orow = p.o + (((int64_t)b * p.H + h) * p.Lq + (int64_t)i * BLK + row) * D;
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
  if (warp == 5) tmem_dealloc(tmem, kTmemCols);
}

template <int D, int BLK>
static int launch_one(const AttnParams &ap, const BatchMeta &meta, const CUtensorMap &tm_q, const CUtensorMap &tm_k_full,
                      const CUtensorMap &tm_k_8, const CUtensorMap &tm_v_full, const CUtensorMap &tm_v_8,
                      cudaStream_t st) {
  auto kern = li_sparse_attn_kernel<D, BLK>;
  constexpr int smem = AttnSmem<D, BLK>::kTotal;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return (int)e;
  dim3 grid(ap.Nqb, ap.H, ap.B);
  kern<<<grid, 192, smem, st>>>(ap, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8);
  return (int)cudaGetLastError();
}

int launch_attn(const AttnParams &ap, const BatchMeta &meta, int d, int blk, const CUtensorMap &tm_q,
                const CUtensorMap &tm_k_full, const CUtensorMap &tm_k_8, const CUtensorMap &tm_v_full,
                const CUtensorMap &tm_v_8, cudaStream_t st, int64_t *n_launches) {
  int e;
  if (d == 128 && blk == 128) e = launch_one<128, 128>(ap, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st);
  else if (d == 128 && blk == 64) e = launch_one<128, 64>(ap, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st);
  else if (d == 64 && blk == 128) e = launch_one<64, 128>(ap, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st);
  else e = launch_one<64, 64>(ap, meta, tm_q, tm_k_full, tm_k_8, tm_v_full, tm_v_8, st);
  if (e == 0 && n_launches) *n_launches += 1;
  return e;
}

}  // namespace li
