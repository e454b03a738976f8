/* li.h -- C ABI of libli.so: the AR-aware block-sparse attention hot path of Light Interaction
 * (arXiv 2605.31158, section 3.3) for NVIDIA B200 (sm_100a).
 *
 * Two operations (PAPER.md = /root/reference/PAPER.md, cited by line):
 *   li_block_select : Eq. 9 block mean pooling of Q and of the historical K, per head;
 *                     Eq. 10 score qbar_i . kbar_m / sqrt(d) and Top_{floor(rM)} per query block.
 *   li_sparse_attn  : Eq. 11 context C_i = T U K^curr U S_i (T = optional text tokens), then softmax
 *                     attention of query block i over C_i ("sparse attention core").
 * The KV context is never materialised: K/V rows are read in place from a frame-paged cache through a
 * frame-index list  memory | temporal window | current chunk  (Fig. 2a "reconstruct the KV
 * cache for the current chunk"; PAPER.md:146-151 describes the copies this replaces).
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer unless its name ends in _host.  The caller owns every buffer; the
 *     library never allocates or frees device memory.  Process-wide state: the loaded kernels, a small cache of
 *     encoded TMA descriptors (keyed by address, shape and strides, so a steady-state call does no driver work), the
 *     launch counter, and a thread-local copy of the last CUDA error code.  No environment variable is read.
 *   - Calls are asynchronous on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream) and
 *     never synchronise the device.  Host arrays are consumed before the call returns.
 *   - Return value: LI_OK (0) or a negative LI_ERR_* code.  No C++ exception crosses this boundary.
 *   - bf16 = IEEE bfloat16 bit patterns (uint16).  Strides are in ELEMENTS; the innermost (d) stride is 1;
 *     every other stride must be a multiple of 8 elements and base pointers 16-byte aligned (TMA rules).
 *   - Logical order of one call's context: history token t in [0, L_hist) is row t mod T_f of
 *     page F[t div T_f]; chunk token u in [0, Lq) is row u mod T_f of page F[n_hist + u div T_f].
 *     History, chunk and queries are tiled separately from their own first token into blocks of
 *     block_k / block_k / block_q tokens; only the last block of each grid may be partial.  (3-D blocks: see the
 *     grid_h/grid_w/bt/bh/bw fields of li_problem.)
 *   - There is no CPU fallback and no second backend: without a CUDA device every compute call fails
 *     with LI_ERR_CUDA.
 */
#ifndef LI_H_
#define LI_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LI_VERSION 200          /* major*100 + minor */
#define LI_MAX_CALLS 64         /* max B per call of the library (batch of independent attention calls) */

enum {
  LI_OK = 0,
  LI_ERR_INVALID_ARG = -1,      /* NULL pointer, non-positive size, bad stride/alignment, bad frame list */
  LI_ERR_UNSUPPORTED = -2,      /* d not in {64,128}; block not in {64,128}; block_q != block_k; B > LI_MAX_CALLS */
  LI_ERR_WORKSPACE   = -3,      /* workspace NULL or smaller than li_workspace_bytes() */
  LI_ERR_CUDA        = -4,      /* a CUDA runtime/driver call failed (no device, launch error, ...); the runtime's own
                                   code is returned by li_last_cuda_error() */
  LI_ERR_TOO_LARGE   = -5       /* li_block_select_static: the problem needs more than LI_STATIC_SCRATCH_BYTES of scratch */
};

/* li_problem.flags */
#define LI_FLAG_NO_SPLIT 1u     /* li_sparse_attn: never split the query blocks of the last wave */
#define LI_FLAG_KV_FP8   2u     /* k_cache / v_cache hold FP8 E4M3 codes, see k_scale / v_scale below */

typedef struct li_problem {
  int32_t B, H, Lq, d;          /* B independent calls; Lq = n_cur_frames * frame_tokens when n_cur_frames > 0 */
  int32_t frame_tokens;         /* T_f, tokens per cache page; multiple of 8 */
  int32_t block_q, block_k;     /* 64 or 128; block_q == block_k */
  int32_t n_pages;              /* pages in the cache pool */
  const void *q;                /* bf16 Q[B,H,Lq,d] */
  int64_t q_sb, q_sh, q_st;     /* batch / head / token strides of Q */
  const void *k_cache;          /* bf16 [n_pages,H,T_f,d] (strides below) */
  const void *v_cache;          /* bf16, same shape and strides as k_cache */
  int64_t kv_sp, kv_sh, kv_st;  /* page / head / token strides of both caches */
  const int32_t *frame_idx;     /* DEVICE int32: concatenated frame lists, logical order mem | win | cur */
  const int32_t *frame_off_host;/* HOST int32 [B+1]: call b owns frame_idx[frame_off[b] .. frame_off[b+1]) */
  int32_t n_cur_frames;         /* the last n_cur_frames entries of every list are the current chunk (>= 0) */
  float   softmax_scale;        /* 0 => 1/sqrt(d) */
  /* 3-D block tiling ("non-overlapping 3D blocks of size (B_t,B_h,B_w)", :321 (4,8,4)/(4,4,8), volume
   * 128).  All five zero = 1-D blocks of block_k consecutive logical tokens.  Otherwise a frame is a grid_h x grid_w
   * row-major grid (frame_tokens == grid_h*grid_w, token = y*grid_w + x) and a region of n frames (history, chunk,
   * queries) is tiled by groups of bt consecutive frames x bh rows x bw columns; block index
   * m = (tg*ceil(grid_h/bh) + hb)*ceil(grid_w/bw) + wb.  Border blocks (grid_h % bh != 0, grid_w % bw != 0) and the last
   * temporal group may be partial: padding never enters a mean nor the softmax, and is never stored (PAPER.md:148,
   * :151).  Both of the paper's geometries run on the 30 x 52 grid: (4,8,4) and (4,4,8).
   * Supported: bt*bh*bw == block_q == block_k, bh*bw == 32, Q contiguous over (B,H) (q_sb == H*q_sh). */
  int32_t grid_h, grid_w;
  int32_t bt, bh, bw;
  /* Text-conditioning tokens T of Eq. 11 (C_i = T U K^curr U S_i; "the model retains all
   * text-conditioning tokens"): a dense, non-paged K/V region attended by every query, never pooled nor
   * selected.  Lt == 0 (and NULL pointers) = no text. */
  int32_t Lt;                   /* text tokens per call */
  const void *text_k;           /* bf16 [B,H,Lt,d] */
  const void *text_v;           /* bf16, same shape and strides */
  int64_t t_sb, t_sh, t_st;     /* batch / head / token strides of both */
  uint32_t flags;               /* LI_FLAG_* bits, 0 = defaults */
  /* FP8 K/V pages (LI_FLAG_KV_FP8; the paper states no cache precision): k_cache and
   * v_cache are uint8 [n_pages,H,T_f,d] of OCP FP8 E4M3 codes (1-4-3, bias 7, no infinities, max 448), strides in
   * elements (= bytes, multiples of 16), value = decode(code) * scale[h] with one fp32 scale per head.  Pages are written
   * by li_quantize_pages.  li_block_select pools the dequantised K; li_sparse_attn replaces every query row by its own
   * e4m3 image (scale max|q_u| / 448, fp32) and runs both contractions on the FP8 tensor-core path, the probabilities
   * rounded to e4m3.  Supported: d == 128, block 128, no text prefix, 1-D or 3-D blocks; li_pool_pages /
   * li_block_select_cached are bf16-only. */
  const float *k_scale;         /* DEVICE fp32 [H] */
  const float *v_scale;         /* DEVICE fp32 [H] */
} li_problem;

/* Eq. 9-10.  For every call b, head h and query block i: pooled means (true cardinality
 * in partial blocks), scores s_{i,m} = qbar_i . kbar_m / sqrt(d) in fp32, and the k_b = min(M_b, top_k_host[b])
 * historical blocks with the largest score (ties -> lowest block index), written in ASCENDING block order.
 *   top_k_host : HOST int32 [B]; the caller computes floor(r*M_b) in integer arithmetic.
 *   kmax       : row pitch of sel_idx, >= max_b k_b and >= 1.
 *   sel_idx    : int32 [B,H,Nqb,kmax]; entries beyond k_b are set to -1.
 *   sel_cnt    : int32 [B,H,Nqb]      = k_b.
 *   scores_opt : NULL, or fp32 [B,H,Nqb,score_pitch] receiving the scores (score_pitch >= max_b M_b).
 *   workspace  : >= li_workspace_bytes(p, kmax) bytes, 256-byte aligned; holds qbar/kbar (fp32).
 * Degenerate cases: M_b == 0 or k_b == 0 give sel_cnt = 0. */
int li_block_select(const li_problem *p, const int32_t *top_k_host, int32_t kmax,
                    int32_t *sel_idx, int32_t *sel_cnt, float *scores_opt, int32_t score_pitch,
                    void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Same as li_block_select, but the pooled historical keys kbar are NOT recomputed: `workspace` must still hold them
 * from an earlier li_block_select on the same history (same frame lists, same K pages, same tiling).  Within one
 * chunk the historical K of a layer does not change across the K denoising steps (the context
 * is reconstructed once per chunk), so only Q has to be pooled again: the call reads Lq*d*2*H bytes instead of
 * (Lq + L_hist)*d*2*H. */
int li_block_select_reuse_kbar(const li_problem *p, const int32_t *top_k_host, int32_t kmax,
                               int32_t *sel_idx, int32_t *sel_cnt, float *scores_opt, int32_t score_pitch,
                               void *workspace, size_t workspace_bytes, void *cuda_stream);

/* li_block_select for callers that cannot allocate device memory (code under CUDA graph capture, serving loops and
 * harnesses that forbid cudaMalloc): same operation, same arguments, same results bit for bit (Eq. 9-10,
 * PAPER.md:131-140), but the scratch (pooled means qbar / kbar, and the score keys of the M > 512 path) lives in a
 * file-scope __device__ array of LI_STATIC_SCRATCH_BYTES inside libli.so instead of a caller-supplied workspace.  The
 * call allocates nothing (no cudaMalloc / cudaFree, no allocating library routine); every GPU that loads the library
 * holds the array until the process exits.
 *   - A problem whose select scratch, align256(B*H*Nqb*d*4) + align256(B*H*Mp*d*4) + align256(B*H*Nqb*max(Mmax,1)*4)
 *     bytes (Mp = Mmax rounded up to 32; li_static_scratch_needed() returns it), exceeds LI_STATIC_SCRATCH_BYTES is
 *     rejected with LI_ERR_TOO_LARGE before anything is launched (`mid` needs 3.7 MB, `long` 7.5 MB).
 *   - ALL calls on a device share the one array, and it keeps the previous call's contents.  Nothing in it has to start
 *     at zero: every value a call reads it has written itself (padding columns of kbar are copied but never used).
 *     Calls that may overlap on the GPU (different streams, no ordering between them) RACE on it: order them, or give
 *     the overlapping ones their own workspace through li_block_select.
 *   - The pooled keys are not kept for li_block_select_reuse_kbar (that call takes the caller's workspace). */
#define LI_STATIC_SCRATCH_BYTES (16u << 20)
int li_block_select_static(const li_problem *p, const int32_t *top_k_host, int32_t kmax,
                           int32_t *sel_idx, int32_t *sel_cnt, float *scores_opt, int32_t score_pitch,
                           void *cuda_stream);
/* Bytes of the array the call above would use for problem p (0 on invalid p); no device is touched. */
size_t li_static_scratch_needed(const li_problem *p);

/* Page-resident pooled slices (3-D tiling only; LI_ERR_UNSUPPORTED otherwise).  A 3-D block is bt frames
 * x one bh x bw patch of the frame grid, and the sum of a frame's K rows over a patch does not depend on where the frame
 * sits in a call's frame list.  li_pool_pages computes these sums for the listed pages (call it for a page whenever its
 * K rows were written: once per chunk for the chunk's pages) into
 *   slice_cache : fp32 [n_pages][H][Hb*Wb][d], li_slice_cache_bytes(p) bytes, 16-byte aligned, owned by the caller;
 * li_block_select_cached is li_block_select with the pooled historical keys (Eq. 9) formed from <= bt cached rows per
 * block instead of the block's 128 K rows: it reads Lq*d*2*H + M*bt*d*4*H bytes instead of (Lq + L_hist)*d*2*H.  Same
 * means up to the fp32 summation order (patch sums first), same scores / top-k semantics.  Every page of the history
 * must have been pooled since it was last written (not checked).  pages_dev: DEVICE int32 [n_list]. */
size_t li_slice_cache_bytes(const li_problem *p);
int li_pool_pages(const li_problem *p, const int32_t *pages_dev, int32_t n_list, float *slice_cache, void *cuda_stream);
int li_block_select_cached(const li_problem *p, const int32_t *top_k_host, int32_t kmax,
                           int32_t *sel_idx, int32_t *sel_cnt, float *scores_opt, int32_t score_pitch,
                           const float *slice_cache, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Eq. 11 + attention.  Query block i of (b,h) attends ALL text tokens (if any), ALL chunk tokens
 * (bidirectional inside the chunk) plus the valid tokens of historical blocks sel_idx[b,h,i,0..sel_cnt[b,h,i]); the same
 * indices address K and V.  softmax in fp32 (online), bf16 tcgen05 MMAs with fp32 accumulation.
 *   o       : bf16 [B,H,Lq,d], contiguous.
 *   lse_opt : NULL or fp32 [B,H,Lq]: log sum_n exp(scale * q.k_n) (natural log).
 * An empty context (no chunk and no selected block) gives o = 0, lse = -inf.
 * sel_idx rows are SETS: the first sel_cnt entries of a row must be distinct values in [0, M_b), in ANY order (the
 * blocks are attended in the order given; li_block_select writes them ascending); sel_cnt <= kmax.  Neither is checked
 * by this call (device data): li_validate checks them on the device.
 *   workspace : optional.  With >= li_workspace_bytes(p, kmax) bytes (256-byte aligned; the same buffer li_block_select
 *               used: its pooled keys are left intact) the kernel may split the query blocks of a sparsely filled last
 *               wave of CTAs across several CTAs and merge their partial results with a second, small launch
 *               (results equal up to fp32 rounding of the merge).  NULL or a smaller buffer: never split. */
int li_sparse_attn(const li_problem *p, const int32_t *sel_idx, const int32_t *sel_cnt, int32_t kmax,
                   void *o, float *lse_opt, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Quantise-on-write for FP8 pages (LI_FLAG_KV_FP8 must be set in p): for t in [0, n_list) page pages_dev[t] of
 * p->k_cache / p->v_cache receives encode(src[t] / scale[h]) -- division in fp32, round to nearest even, saturating at
 * +-448 (PTX cvt.rn.satfinite.e4m3x2.f32) -- of the bf16 rows k_src / v_src [n_list,H,T_f,d] (contiguous, 16-byte
 * aligned).  HBM-bound: reads 4 and writes 2 bytes per element pair.  Page ids outside [0, n_pages) are skipped. */
int li_quantize_pages(const li_problem *p, const void *k_src, const void *v_src, const int32_t *pages_dev, int32_t n_list,
                      void *cuda_stream);

/* Debug validation of DEVICE-side inputs that the calls above trust (one small launch, asynchronous, no host
 * synchronisation; meant for debug builds of the caller, not for the hot loop):
 *   - every page id of every call's frame list lies in [0, n_pages)                                   LI_BAD_PAGE_ID
 *   - when sel_idx/sel_cnt are given (both or neither): 0 <= sel_cnt <= min(kmax, M_b)                LI_BAD_SEL_CNT
 *     every one of the first sel_cnt entries lies in [0, M_b)                                         LI_BAD_SEL_RANGE
 *     and the entries of a row are distinct (checked for M_b <= 262144)                               LI_BAD_SEL_DUPLICATE
 * error_dev: DEVICE int32[4], overwritten: [0] = OR of the LI_BAD_* bits found (0 = all good), [1] = call b,
 * [2] = position (frame-list entry, or flat (h*Nqb + i)*kmax + t) and [3] = value of ONE offender (the lowest bit's
 * first-arriving report; which one is unspecified when several exist).  Without it a bad page id is an out-of-bounds
 * read in li_block_select and a silently zero-filled tile in li_sparse_attn. */
#define LI_BAD_PAGE_ID 1
#define LI_BAD_SEL_CNT 2
#define LI_BAD_SEL_RANGE 4
#define LI_BAD_SEL_DUPLICATE 8
int li_validate(const li_problem *p, const int32_t *sel_idx, const int32_t *sel_cnt, int32_t kmax,
                int32_t *error_dev, void *cuda_stream);

/* Bytes of workspace the calls above need for problem p (0 on invalid p): li_block_select's pooled means and score keys,
 * followed by the partial-result buffers of li_sparse_attn's split (a fixed ~21 MB at d = 128). */
size_t li_workspace_bytes(const li_problem *p, int32_t kmax);

/* Adaptive context management and the frame list it produces -- what li_problem.frame_idx is built from,
 * once per chunk.  All pointers are DEVICE pointers; nothing is read back by the call.
 *   Eq. 1  D_t    = mean over all n_latent dimensions of (z_prev1 - z_prev2)^2         (fp32 products, fp64 sums)
 *   Eq. 2  Dbar_t = alpha D_t + (1 - alpha) Dbar_{t-1}; ema_state = {Dbar, valid}: valid == 0 -> Dbar_t = D_t; updated
 *          in place (fp32)
 *   Eq. 3  L_t    = clip([L_max * kappa / (Dbar_t + kappa)], 1, L_max) in fp32, evaluated as (L_max*kappa)/(Dbar_t+kappa);
 *          the bracket (garbled in the paper) is floor, or round-half-to-even when round_nearest != 0
 *   Eq. 4  keep_memory = !(max_j s_pose[j] < tau_pose); no candidate (n_cand == 0) -> 0
 *   frame_idx_out = [mem_pages[0..n_mem) if keep_memory] + [the min(L_t, n_win) LAST entries of win_pages (oldest ->
 *          newest)] + [cur_pages[0..n_cur)]. */
typedef struct li_policy {
  const void *z_prev1;          /* latents of the two most recent stable units, 16-byte aligned */
  const void *z_prev2;
  int64_t n_latent;             /* elements of each */
  int32_t latent_bf16;          /* 0: fp32, 1: bf16 */
  float alpha;                  /* in (0, 1] */
  float kappa;                  /* > 0 */
  int32_t L_max;                /* L_m of Eq. 3, >= 1 */
  int32_t round_nearest;        /* Eq. 3 bracket: 0 floor, 1 nearest */
  float *ema_state;             /* float[2] */
  const float *s_pose;          /* fp32 [n_cand] (may be NULL when n_cand == 0) */
  int32_t n_cand;
  float tau_pose;
  const int32_t *mem_pages;     /* int32 [n_mem] */
  int32_t n_mem;
  const int32_t *win_pages;     /* int32 [n_win] */
  int32_t n_win;
  const int32_t *cur_pages;     /* int32 [n_cur] */
  int32_t n_cur;
} li_policy;

typedef struct li_policy_result {   /* written to DEVICE memory by li_context_policy */
  float D_t, D_bar;
  int32_t L_t, keep_memory;
  int32_t n_hist_frames;        /* (kept memory) + (window frames used) */
  int32_t n_frames;             /* entries written to frame_idx_out = n_hist_frames + n_cur */
} li_policy_result;

/* frame_idx_capacity must be >= n_mem + min(L_max, n_win) + n_cur (entries past n_frames are left untouched);
 * workspace >= li_policy_workspace_bytes() bytes, 256-byte aligned.  Two kernel launches, no host synchronisation: the
 * caller reads result_dev back (24 bytes) when it needs the frame count on the host (li_problem.frame_off_host). */
int li_context_policy(const li_policy *pp, int32_t *frame_idx_out, int32_t frame_idx_capacity,
                      li_policy_result *result_dev, void *workspace, size_t workspace_bytes, void *cuda_stream);
size_t li_policy_workspace_bytes(void);

/* Number of kernel launches the calls above issued since the last li_reset_launch_count()
 * (bench.py's gpu_launches). */
int64_t li_launch_count(void);
void li_reset_launch_count(void);

const char *li_strerror(int code);
int li_version(void);
/* cudaError_t of the last call of THIS thread that returned LI_ERR_CUDA (0 if none). */
int li_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LI_H_ */
