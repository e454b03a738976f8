// li_internal.h -- kernel parameter blocks shared by the C-ABI layer (li_api.cu) and the kernels.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/li.h"

namespace li {

// Per-launch description of the batch (passed by value as a kernel parameter: no device-side metadata copy).
struct BatchMeta {
  int32_t frame_off[LI_MAX_CALLS + 1];  // CSR offsets into frame_idx
  int32_t top_k[LI_MAX_CALLS];          // k_b already clamped to M_b (select only)
};

// Block tiling of a region of n frames.  bt == 0: 1-D blocks of `blk` consecutive logical tokens.  Otherwise 3-D blocks
// of bt frames x bh rows x bw columns of the gh x gw frame grid, block index
// m = (tg*Hb + hb)*Wb + wb; a block's rows are ordered (frame, y, x), 32 = bh*bw rows per frame slice.
struct Tiling {
  int32_t gh, gw, bt, bh, bw, Hb, Wb;
  int32_t bw_log2;                       // bh * bw == 32, so bw is a power of two
  __host__ __device__ int num_blocks(int n_frames, int T_f, int blk) const {
    return bt > 0 ? ((n_frames + bt - 1) / bt) * Hb * Wb : (n_frames * T_f + blk - 1) / blk;
  }
};

struct SelectParams {
  Tiling tl;
  int32_t skip_k;   // 1: kbar in the workspace is still valid (li_block_select_reuse_kbar): pool Q only
  int32_t B, H, Lq, d, T_f, blk, n_cur, Nqb, Mmax, Mp, kmax, score_pitch;   // Mp = Mmax rounded up to 32
  int32_t n_pages;  // page ids outside [0, n_pages) are never dereferenced (their rows count as zeros; li_validate reports them)
  const uint16_t *q;
  int64_t q_sb, q_sh, q_st;
  const uint16_t *k_cache;
  int64_t kv_sp, kv_sh, kv_st;
  const int32_t *frame_idx;
  float *qbar;     // [B,H,Nqb,d]
  float *kbar;     // [B,H,d,Mp]  (transposed: channel-major)
  uint32_t *keys;  // [B,H,Nqb,Mmax] order-preserving score keys
  int32_t *sel_idx;
  int32_t *sel_cnt;
  float *scores;   // optional
  float inv_sqrt_d;
  const float *slice_cache;   // 3-D tiling: per-page patch sums [n_pages,H,Hb*Wb,d]; non-null: kbar is formed from them
  const float *k_scale;       // LI_FLAG_KV_FP8: k_cache holds e4m3 codes (byte strides), value = decode * k_scale[h]
};

struct AttnParams {
  Tiling tl;
  int32_t B, H, Lq, T_f, n_cur, Nqb, Nc, kmax;
  int32_t Lt;             // text tokens (T of Eq. 11), 0 = none
  int32_t has_box_full;   // 1: tensor maps with a full half-tile box exist (T_f >= block/2)
  int32_t no_split;       // LI_FLAG_NO_SPLIT
  float scale_log2;       // softmax_scale * log2(e)
  const int32_t *frame_idx;
  const int32_t *sel_idx;
  const int32_t *sel_cnt;
  uint16_t *o;
  float *lse;
  const float *k_scale, *v_scale;   // LI_FLAG_KV_FP8: per-head scales of the e4m3 K / V pages (else null)
  // tail-wave split: CTAs [0, split_first) own a whole query block each; from split_first on, n_split
  // consecutive CTAs share one query block, each taking a contiguous range of its half-tiles and writing unnormalised
  // partial results, which li_attn_combine_kernel merges.  n_split == 1: no split (split_first == number of blocks).
  int32_t split_first, n_split;
  float *part_o;    // [slot][128 rows][d] fp32, slot = CTA - split_first
  float2 *part_ml;  // [slot][128 rows] (reference maximum in log2 units, row sum)
};

constexpr int kMaxSplitSlots = 320;   // upper bound of split CTAs (<= 2 CTAs per SM), sizes the workspace

// multiprocessors of the current device, queried once per device (0 if the query fails); defined in li_api.cu
int device_sm_count();

// launches (defined in the .cu files); return cudaError_t as int
int launch_select(const SelectParams &sp, const BatchMeta &meta, cudaStream_t st, int64_t *n_launches);
// FP8 pages (li_fp8.cu): pooling of the historical K blocks from e4m3 pages; quantise-on-write
int launch_pool_k8(const SelectParams &sp, const BatchMeta &meta, cudaStream_t st, int64_t *n_launches);
struct QuantParams {
  int32_t H, T_f, d, n_pages;
  const uint16_t *k_src, *v_src;      // bf16 [n_list,H,T_f,d]
  uint8_t *k_cache, *v_cache;
  int64_t kv_sp, kv_sh, kv_st;
  const float *k_scale, *v_scale;
  const int32_t *pages;
};
int launch_quantize_pages(const QuantParams &qp, int n_list, cudaStream_t st, int64_t *n_launches);
int launch_pool_pages(const SelectParams &sp, const int32_t *pages, int n_list, float *cache, cudaStream_t st, int64_t *n_launches);
int launch_attn(const AttnParams &ap, const BatchMeta &meta, int d, int blk, const CUtensorMap &tm_q,
                const CUtensorMap &tm_tk, const CUtensorMap &tm_tv, const CUtensorMap &tm_k_full, const CUtensorMap &tm_k_8, const CUtensorMap &tm_v_full,
                const CUtensorMap &tm_v_8, cudaStream_t st, int64_t *n_launches);

// li_validate (debug check of device-side inputs, include/li.h)
struct ValidateParams {
  Tiling tl;
  int32_t B, H, Nqb, T_f, blk, n_cur, n_pages, kmax, Mmax;
  const int32_t *frame_idx;
  const int32_t *sel_idx;   // may be null (frame lists only)
  const int32_t *sel_cnt;
  int32_t *err;             // int32[4], zeroed before the launch
};
int launch_validate(const ValidateParams &vp, const BatchMeta &meta, cudaStream_t st, int64_t *n_launches);

int launch_policy(const li_policy &pp, int32_t *frame_idx_out, li_policy_result *result, double *partial, cudaStream_t st,
                  int64_t *n_launches);
constexpr size_t kPolicyWorkspaceBytes = 1024 * sizeof(double);   // one fp64 partial sum per CTA of li_mse_partial_kernel

}  // namespace li
