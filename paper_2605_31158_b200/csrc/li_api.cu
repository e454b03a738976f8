// li_api.cu -- the C ABI of libli.so (include/li.h): argument validation, workspace carving, TMA tensor-map
// encoding and kernel launches.  No device allocation, no synchronisation, no environment variable.  Process-wide
// state: the launch counter, the lazily resolved cuTensorMapEncodeTiled entry point, a small cache of encoded tensor
// maps (a steady-state call does no driver work) and a thread-local copy of the last CUDA error code.
#include <atomic>
#include <cmath>
#include <cstring>
#include <mutex>

#include "li_internal.h"

namespace li {
int device_sm_count() {
  static std::atomic<int> sm_count[64];
  int dev = 0, n_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  n_sm = sm_count[dev & 63].load(std::memory_order_relaxed);
  if (n_sm == 0 && cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess)
    sm_count[dev & 63].store(n_sm, std::memory_order_relaxed);
  return n_sm;
}
}  // namespace li

namespace {

std::atomic<int64_t> g_launches{0};
thread_local int t_last_cuda_error = 0;

int cuda_failed(int e) {
  t_last_cuda_error = e;
  return LI_ERR_CUDA;
}

using EncodeFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                              const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                              CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeFn get_encode() {
  static std::atomic<void *> cached{nullptr};
  void *fn = cached.load();
  if (fn == nullptr) {
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
      return nullptr;
    cached.store(fn);
  }
  return reinterpret_cast<EncodeFn>(fn);
}

// Encoded tensor maps are pure functions of (address, shape, strides, box): they are cached, so that a call with the
// same tensors as an earlier one (the steady state of an AR loop) does no driver work.
struct MapKey {
  const void *base;
  int32_t rank, d, box[4], elem_bytes;   // elem_bytes: 2 = bf16 (inner box 64 elements), 1 = FP8 codes (inner box 128)
  int64_t dims[4], strides[4];
  bool operator==(const MapKey &o) const { return std::memcmp(this, &o, sizeof(MapKey)) == 0; }
};
struct MapCache {
  static constexpr int kEntries = 64;
  std::mutex mu;
  MapKey keys[kEntries];
  CUtensorMap maps[kEntries];
  int used = 0, next = 0;
};
MapCache g_maps;

bool encode_cached(CUtensorMap *tm, const MapKey &key) {
  {
    std::lock_guard<std::mutex> lock(g_maps.mu);
    for (int e = 0; e < g_maps.used; ++e)
      if (g_maps.keys[e] == key) { *tm = g_maps.maps[e]; return true; }
  }
  EncodeFn enc = get_encode();
  if (enc == nullptr) return false;
  cuuint64_t dims[5] = {(cuuint64_t)key.d};
  cuuint64_t strides[4];
  cuuint32_t box[5] = {(cuuint32_t)(128 / key.elem_bytes)}, estr[5] = {1, 1, 1, 1, 1};   // 128 bytes = the swizzle span
  for (int k = 0; k + 1 < key.rank; ++k) {
    dims[k + 1] = (cuuint64_t)key.dims[k];
    strides[k] = (cuuint64_t)key.strides[k] * key.elem_bytes;
    box[k + 1] = (cuuint32_t)key.box[k];
  }
  CUresult r = enc(tm, key.elem_bytes == 1 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16,
                   (cuuint32_t)key.rank, const_cast<void *>(key.base), dims, strides, box,
                   estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  std::lock_guard<std::mutex> lock(g_maps.mu);
  const int slot = g_maps.used < MapCache::kEntries ? g_maps.used++ : (g_maps.next++ % MapCache::kEntries);
  g_maps.keys[slot] = key;
  g_maps.maps[slot] = *tm;
  return true;
}

// bf16 tensor [n3, n2, n1, d] (innermost first: d, n1, n2, n3), strides in elements, box = 64 x rows x 1 x 1,
// SWIZZLE_128B, out-of-bounds elements read as zero.
bool encode_map(CUtensorMap *tm, const void *base, int d, int64_t n1, int64_t n2, int64_t n3, int64_t s1, int64_t s2,
                int64_t s3, int box_rows, int elem_bytes = 2) {
  MapKey k;
  std::memset(&k, 0, sizeof(k));
  k.base = base; k.rank = 4; k.d = d; k.elem_bytes = elem_bytes;
  k.dims[0] = n1; k.dims[1] = n2; k.dims[2] = n3;
  k.strides[0] = s1; k.strides[1] = s2; k.strides[2] = s3;
  k.box[0] = box_rows; k.box[1] = 1; k.box[2] = 1;
  return encode_cached(tm, k);
}

// bf16 tensor viewed as 5-D [n4, n3, gh, gw, d] (innermost first: d, gw, gh, n3, n4), box = 64 x bw x bh x 1 x 1:
// one frame's bh x bw patch of a 3-D block = 32 rows of 128 bytes, SWIZZLE_128B, zero fill outside.
bool encode_map5(CUtensorMap *tm, const void *base, int d, int gw, int gh, int64_t n3, int64_t n4, int64_t s_w,
                 int64_t s_h, int64_t s3, int64_t s4, int bw, int bh, int elem_bytes = 2) {
  MapKey k;
  std::memset(&k, 0, sizeof(k));
  k.base = base; k.rank = 5; k.d = d; k.elem_bytes = elem_bytes;
  k.dims[0] = gw; k.dims[1] = gh; k.dims[2] = n3; k.dims[3] = n4;
  k.strides[0] = s_w; k.strides[1] = s_h; k.strides[2] = s3; k.strides[3] = s4;
  k.box[0] = bw; k.box[1] = bh; k.box[2] = 1; k.box[3] = 1;
  return encode_cached(tm, k);
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }
inline size_t mpad(int m) { return m > 0 ? (size_t)((m + 31) & ~31) : 32; }   // row pitch of the transposed kbar

struct Derived {
  int Nqb, Nc, Mmax;
  li::Tiling tl;
  li::BatchMeta meta;
};

// Validates p and fills the derived integers.  Returns LI_OK or an error code.  pages_only: the call touches only the
// K cache and the tiling (li_pool_pages, li_slice_cache_bytes): Q, the frame lists and the text region are not looked at.
int check_problem(const li_problem *p, Derived *dv, bool pages_only = false) {
  if (p == nullptr) return LI_ERR_INVALID_ARG;
  if (pages_only) {
    if (p->H <= 0 || p->frame_tokens <= 0 || p->n_pages <= 0) return LI_ERR_INVALID_ARG;
    if (p->d != 64 && p->d != 128) return LI_ERR_UNSUPPORTED;
    if (p->block_k != 64 && p->block_k != 128) return LI_ERR_UNSUPPORTED;
    if (p->frame_tokens % 8 != 0 || p->k_cache == nullptr || ((uintptr_t)p->k_cache & 15u)) return LI_ERR_INVALID_ARG;
    const int64_t ks[3] = {p->kv_sp, p->kv_sh, p->kv_st};
    for (int64_t s : ks)
      if (s <= 0 || s % 8 != 0) return LI_ERR_INVALID_ARG;
    if (p->kv_st < p->d) return LI_ERR_INVALID_ARG;
    std::memset(&dv->meta, 0, sizeof(dv->meta));
    std::memset(&dv->tl, 0, sizeof(dv->tl));
    if (p->grid_h <= 0 || p->grid_w <= 0 || p->bt <= 0 || p->bh <= 0 || p->bw <= 0) return LI_ERR_UNSUPPORTED;
    if (p->grid_h * p->grid_w != p->frame_tokens) return LI_ERR_INVALID_ARG;
    if (p->bt * p->bh * p->bw != p->block_k || p->bh * p->bw != 32) return LI_ERR_UNSUPPORTED;
    dv->tl.gh = p->grid_h; dv->tl.gw = p->grid_w; dv->tl.bt = p->bt; dv->tl.bh = p->bh; dv->tl.bw = p->bw;
    dv->tl.Hb = (p->grid_h + p->bh - 1) / p->bh; dv->tl.Wb = (p->grid_w + p->bw - 1) / p->bw;
    for (dv->tl.bw_log2 = 0; (1 << dv->tl.bw_log2) < p->bw; ++dv->tl.bw_log2) {}
    dv->Nqb = dv->Nc = dv->Mmax = 0;
    return LI_OK;
  }
  if (p->B <= 0 || p->H <= 0 || p->Lq <= 0 || p->frame_tokens <= 0 || p->n_pages <= 0 || p->n_cur_frames < 0)
    return LI_ERR_INVALID_ARG;
  if (p->d != 64 && p->d != 128) return LI_ERR_UNSUPPORTED;
  if (p->block_q != p->block_k || (p->block_k != 64 && p->block_k != 128)) return LI_ERR_UNSUPPORTED;
  if (p->B > LI_MAX_CALLS) return LI_ERR_UNSUPPORTED;
  if (p->frame_tokens % 8 != 0) return LI_ERR_INVALID_ARG;
  if (p->q == nullptr || p->k_cache == nullptr || p->v_cache == nullptr || p->frame_idx == nullptr ||
      p->frame_off_host == nullptr)
    return LI_ERR_INVALID_ARG;
  if (p->n_cur_frames > 0 && p->Lq != p->n_cur_frames * p->frame_tokens) return LI_ERR_INVALID_ARG;
  if (p->softmax_scale < 0.f || !std::isfinite(p->softmax_scale)) return LI_ERR_INVALID_ARG;
  const int64_t strides[6] = {p->q_sb, p->q_sh, p->q_st, p->kv_sp, p->kv_sh, p->kv_st};
  for (int64_t s : strides)
    if (s <= 0 || s % 8 != 0) return LI_ERR_INVALID_ARG;
  if (p->q_st < p->d || p->kv_st < p->d) return LI_ERR_INVALID_ARG;
  if (((uintptr_t)p->q | (uintptr_t)p->k_cache | (uintptr_t)p->v_cache) & 15u) return LI_ERR_INVALID_ARG;
  if (p->flags & LI_FLAG_KV_FP8) {
    if (p->d != 128 || p->block_k != 128 || p->Lt != 0) return LI_ERR_UNSUPPORTED;
    if (p->k_scale == nullptr || p->v_scale == nullptr) return LI_ERR_INVALID_ARG;
    if (p->kv_sp % 16 != 0 || p->kv_sh % 16 != 0 || p->kv_st % 16 != 0) return LI_ERR_INVALID_ARG;   // byte strides (TMA: 16)
  }
  if (p->Lt < 0) return LI_ERR_INVALID_ARG;
  if (p->Lt > 0) {
    if (p->text_k == nullptr || p->text_v == nullptr) return LI_ERR_INVALID_ARG;
    if ((((uintptr_t)p->text_k | (uintptr_t)p->text_v) & 15u) != 0) return LI_ERR_INVALID_ARG;
    const int64_t ts[3] = {p->t_sb, p->t_sh, p->t_st};
    for (int64_t s : ts)
      if (s <= 0 || s % 8 != 0) return LI_ERR_INVALID_ARG;
    if (p->t_st < p->d) return LI_ERR_INVALID_ARG;
  }
  std::memset(&dv->meta, 0, sizeof(dv->meta));
  std::memset(&dv->tl, 0, sizeof(dv->tl));
  const bool any3d = p->grid_h | p->grid_w | p->bt | p->bh | p->bw;
  if (any3d) {
    if (p->grid_h <= 0 || p->grid_w <= 0 || p->bt <= 0 || p->bh <= 0 || p->bw <= 0) return LI_ERR_INVALID_ARG;
    if (p->grid_h * p->grid_w != p->frame_tokens) return LI_ERR_INVALID_ARG;
    if (p->Lq % p->frame_tokens != 0) return LI_ERR_INVALID_ARG;
    if (p->bt * p->bh * p->bw != p->block_k || p->bh * p->bw != 32) return LI_ERR_UNSUPPORTED;
    if (p->q_sb != (int64_t)p->H * p->q_sh && p->B > 1) return LI_ERR_UNSUPPORTED;
    dv->tl.gh = p->grid_h; dv->tl.gw = p->grid_w; dv->tl.bt = p->bt; dv->tl.bh = p->bh; dv->tl.bw = p->bw;
    dv->tl.Hb = (p->grid_h + p->bh - 1) / p->bh; dv->tl.Wb = (p->grid_w + p->bw - 1) / p->bw;
    for (dv->tl.bw_log2 = 0; (1 << dv->tl.bw_log2) < p->bw; ++dv->tl.bw_log2) {}
  }
  int mmax = 0;
  if (p->frame_off_host[0] < 0) return LI_ERR_INVALID_ARG;
  for (int b = 0; b < p->B; ++b) {
    const int n = p->frame_off_host[b + 1] - p->frame_off_host[b];
    if (n < p->n_cur_frames) return LI_ERR_INVALID_ARG;
    const int64_t L_hist = (int64_t)(n - p->n_cur_frames) * p->frame_tokens;
    if (L_hist + p->Lq > (int64_t)1 << 30) return LI_ERR_INVALID_ARG;
    const int M = dv->tl.num_blocks(n - p->n_cur_frames, p->frame_tokens, p->block_k);
    if (M > mmax) mmax = M;
  }
  for (int b = 0; b <= p->B; ++b) dv->meta.frame_off[b] = p->frame_off_host[b];
  dv->Nqb = any3d ? dv->tl.num_blocks(p->Lq / p->frame_tokens, p->frame_tokens, p->block_q)
                  : (p->Lq + p->block_q - 1) / p->block_q;
  dv->Nc = dv->tl.num_blocks(p->n_cur_frames, p->frame_tokens, p->block_k);
  dv->Mmax = mmax;
  return LI_OK;
}

size_t ws_bytes(const li_problem *p, const Derived &dv) {
  const size_t qbar = align256((size_t)p->B * p->H * dv.Nqb * p->d * 4);
  const size_t kbar = align256((size_t)p->B * p->H * mpad(dv.Mmax) * p->d * 4);
  const size_t keys = align256((size_t)p->B * p->H * dv.Nqb * (dv.Mmax > 0 ? dv.Mmax : 1) * 4);
  return qbar + kbar + keys;
}

// partial results of the attention kernel's tail-wave split: [slots][128 rows][d] fp32 + [slots][128] float2
size_t ws_split_o_bytes(const li_problem *p) { return align256((size_t)li::kMaxSplitSlots * 128 * p->d * 4); }
size_t ws_split_bytes(const li_problem *p) { return ws_split_o_bytes(p) + align256((size_t)li::kMaxSplitSlots * 128 * 8); }

}  // namespace

extern "C" {

size_t li_workspace_bytes(const li_problem *p, int32_t kmax) {
  (void)kmax;
  Derived dv;
  if (check_problem(p, &dv) != LI_OK) return 0;
  return ws_bytes(p, dv) + ws_split_bytes(p);
}

static int block_select_impl(const li_problem *p, const int32_t *top_k_host, int32_t kmax, int32_t *sel_idx,
                             int32_t *sel_cnt, float *scores_opt, int32_t score_pitch, void *workspace,
                             size_t workspace_bytes, void *cuda_stream, int skip_k, const float *slice_cache = nullptr) {
  Derived dv;
  int rc = check_problem(p, &dv);
  if (rc != LI_OK) return rc;
  if (slice_cache != nullptr && dv.tl.bt == 0) return LI_ERR_UNSUPPORTED;   // patch sums exist for 3-D blocks only
  if (slice_cache != nullptr && (p->flags & LI_FLAG_KV_FP8)) return LI_ERR_UNSUPPORTED;   // ... and for bf16 pages only
  if (top_k_host == nullptr || sel_idx == nullptr || sel_cnt == nullptr || kmax < 1) return LI_ERR_INVALID_ARG;
  if (scores_opt != nullptr && score_pitch < dv.Mmax) return LI_ERR_INVALID_ARG;
  if (workspace == nullptr || workspace_bytes < ws_bytes(p, dv) + ws_split_bytes(p) || ((uintptr_t)workspace & 255u))
    return LI_ERR_WORKSPACE;
  for (int b = 0; b < p->B; ++b) {
    if (top_k_host[b] < 0) return LI_ERR_INVALID_ARG;
    const int n_hist = dv.meta.frame_off[b + 1] - dv.meta.frame_off[b] - p->n_cur_frames;
    const int M = dv.tl.num_blocks(n_hist, p->frame_tokens, p->block_k);
    const int k = top_k_host[b] < M ? top_k_host[b] : M;
    if (k > kmax) return LI_ERR_INVALID_ARG;
    dv.meta.top_k[b] = k;
  }

  li::SelectParams sp;
  std::memset(&sp, 0, sizeof(sp));
  sp.tl = dv.tl;
  sp.skip_k = skip_k;
  sp.B = p->B; sp.H = p->H; sp.Lq = p->Lq; sp.d = p->d; sp.T_f = p->frame_tokens; sp.blk = p->block_k;
  sp.n_cur = p->n_cur_frames; sp.Nqb = dv.Nqb; sp.Mmax = dv.Mmax; sp.kmax = kmax; sp.n_pages = p->n_pages;
  sp.score_pitch = score_pitch;
  sp.q = (const uint16_t *)p->q; sp.q_sb = p->q_sb; sp.q_sh = p->q_sh; sp.q_st = p->q_st;
  sp.k_cache = (const uint16_t *)p->k_cache; sp.kv_sp = p->kv_sp; sp.kv_sh = p->kv_sh; sp.kv_st = p->kv_st;
  sp.frame_idx = p->frame_idx;
  sp.qbar = (float *)workspace;
  sp.kbar = (float *)((char *)workspace + align256((size_t)p->B * p->H * dv.Nqb * p->d * 4));
  sp.Mp = (int32_t)mpad(dv.Mmax);
  sp.keys = (uint32_t *)((char *)sp.kbar + align256((size_t)p->B * p->H * mpad(dv.Mmax) * p->d * 4));
  sp.sel_idx = sel_idx; sp.sel_cnt = sel_cnt; sp.scores = scores_opt;
  sp.inv_sqrt_d = 1.0f / std::sqrt((float)p->d);
  int64_t n = 0;
  int e = 0;
  sp.slice_cache = slice_cache;             // non-null: the pool kernel forms kbar from the cached patch sums
  sp.k_scale = (p->flags & LI_FLAG_KV_FP8) ? p->k_scale : nullptr;
  e = li::launch_select(sp, dv.meta, (cudaStream_t)cuda_stream, &n);
  g_launches += n;
  return e == 0 ? LI_OK : cuda_failed(e);
}

size_t li_slice_cache_bytes(const li_problem *p) {
  Derived dv;
  if (check_problem(p, &dv, true) != LI_OK || (p->flags & LI_FLAG_KV_FP8)) return 0;   // bf16 pages only
  return (size_t)p->n_pages * p->H * dv.tl.Hb * dv.tl.Wb * p->d * 4;
}

int li_pool_pages(const li_problem *p, const int32_t *pages_dev, int32_t n_list, float *slice_cache, void *cuda_stream) {
  Derived dv;
  int rc = check_problem(p, &dv, true);
  if (rc != LI_OK) return rc;
  if (p->flags & LI_FLAG_KV_FP8) return LI_ERR_UNSUPPORTED;
  if (n_list < 0 || slice_cache == nullptr || (n_list > 0 && pages_dev == nullptr) || ((uintptr_t)slice_cache & 15u))
    return LI_ERR_INVALID_ARG;
  li::SelectParams sp;
  std::memset(&sp, 0, sizeof(sp));
  sp.tl = dv.tl;
  sp.H = p->H; sp.d = p->d; sp.n_pages = p->n_pages;
  sp.k_cache = (const uint16_t *)p->k_cache; sp.kv_sp = p->kv_sp; sp.kv_sh = p->kv_sh; sp.kv_st = p->kv_st;
  int64_t n = 0;
  const int e = li::launch_pool_pages(sp, pages_dev, n_list, slice_cache, (cudaStream_t)cuda_stream, &n);
  g_launches += n;
  return e == 0 ? LI_OK : cuda_failed(e);
}

int li_block_select_cached(const li_problem *p, const int32_t *top_k_host, int32_t kmax, int32_t *sel_idx,
                           int32_t *sel_cnt, float *scores_opt, int32_t score_pitch, const float *slice_cache,
                           void *workspace, size_t workspace_bytes, void *cuda_stream) {
  if (slice_cache == nullptr) return LI_ERR_INVALID_ARG;
  return block_select_impl(p, top_k_host, kmax, sel_idx, sel_cnt, scores_opt, score_pitch, workspace, workspace_bytes,
                           cuda_stream, 0, slice_cache);
}

int li_block_select(const li_problem *p, const int32_t *top_k_host, int32_t kmax, int32_t *sel_idx, int32_t *sel_cnt,
                    float *scores_opt, int32_t score_pitch, void *workspace, size_t workspace_bytes,
                    void *cuda_stream) {
  return block_select_impl(p, top_k_host, kmax, sel_idx, sel_cnt, scores_opt, score_pitch, workspace, workspace_bytes,
                           cuda_stream, 0);
}

int li_block_select_reuse_kbar(const li_problem *p, const int32_t *top_k_host, int32_t kmax, int32_t *sel_idx,
                               int32_t *sel_cnt, float *scores_opt, int32_t score_pitch, void *workspace,
                               size_t workspace_bytes, void *cuda_stream) {
  return block_select_impl(p, top_k_host, kmax, sel_idx, sel_cnt, scores_opt, score_pitch, workspace, workspace_bytes,
                           cuda_stream, 1);
}

// ----------------------------------------------------------------------------- li_block_select_static (include/li.h)
// Scratch of the no-allocation entry point: one array per device that loads the library, shared by every call, never
// cleared (a call reads only what it has written).  In host code the NAME g_static_scratch is a host-side stand-in, not
// a device address; the address the kernels get is looked up once per device with cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_static_scratch[LI_STATIC_SCRATCH_BYTES];

static int static_scratch_ptr(void **out) {
  static std::atomic<void *> dev_ptr[64];                  // per device ordinal, resolved with that device current
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return (int)e;
  if (dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
  void *ptr = dev_ptr[dev].load(std::memory_order_acquire);
  if (ptr == nullptr) {
    e = cudaGetSymbolAddress(&ptr, g_static_scratch);
    if (e != cudaSuccess) return (int)e;
    if (ptr == nullptr || ((uintptr_t)ptr & 255u)) return (int)cudaErrorInvalidSymbol;
    dev_ptr[dev].store(ptr, std::memory_order_release);
  }
  *out = ptr;
  return 0;
}

size_t li_static_scratch_needed(const li_problem *p) {
  Derived dv;
  if (check_problem(p, &dv) != LI_OK) return 0;
  return ws_bytes(p, dv);
}

int li_block_select_static(const li_problem *p, const int32_t *top_k_host, int32_t kmax, int32_t *sel_idx,
                           int32_t *sel_cnt, float *scores_opt, int32_t score_pitch, void *cuda_stream) {
  Derived dv;
  const int rc = check_problem(p, &dv);
  if (rc != LI_OK) return rc;
  const size_t need = ws_bytes(p, dv);                     // what li_block_select touches of its workspace
  if (need > (size_t)LI_STATIC_SCRATCH_BYTES) return LI_ERR_TOO_LARGE;
  void *scratch = nullptr;
  const int e = static_scratch_ptr(&scratch);
  if (e != 0) return cuda_failed(e);
  // block_select_impl asks for the full li_workspace_bytes (select region + the attention kernel's split region behind
  // it) but reads and writes the select region only, which `need` bounds: the size passed is that requirement
  return block_select_impl(p, top_k_host, kmax, sel_idx, sel_cnt, scores_opt, score_pitch, scratch,
                           need + ws_split_bytes(p), cuda_stream, 0);
}

int li_sparse_attn(const li_problem *p, const int32_t *sel_idx, const int32_t *sel_cnt, int32_t kmax, void *o,
                   float *lse_opt, void *workspace, size_t workspace_bytes, void *cuda_stream) {
  Derived dv;
  int rc = check_problem(p, &dv);
  if (rc != LI_OK) return rc;
  if (sel_idx == nullptr || sel_cnt == nullptr || o == nullptr || kmax < 1) return LI_ERR_INVALID_ARG;
  if ((uintptr_t)o & 15u) return LI_ERR_INVALID_ARG;
  if (workspace != nullptr && ((uintptr_t)workspace & 255u)) return LI_ERR_WORKSPACE;
  // scratch is optional here: only the tail-wave split uses it (its region lies behind li_block_select's, so pooled
  // keys kept for li_block_select_reuse_kbar survive); without a full-size workspace the split is simply not used
  const bool have_ws = workspace != nullptr && workspace_bytes >= ws_bytes(p, dv) + ws_split_bytes(p);

  const int blk = p->block_k;
  const int half = blk / 2;                 // K/V are fetched as half-tiles of blk/2 rows
  const int has_full = p->frame_tokens >= half ? 1 : 0;
  CUtensorMap tm_q, tm_kf, tm_k8, tm_vf, tm_v8;
  bool ok;
  const int eb = (p->flags & LI_FLAG_KV_FP8) ? 1 : 2;      // bytes per K/V element
  if (dv.tl.bt > 0) {
    // 3-D blocks: 5-D maps (d, grid column, grid row, head | frame, page | batch*head)
    const int gw = p->grid_w, gh = p->grid_h;
    ok = encode_map5(&tm_q, p->q, p->d, gw, gh, p->Lq / p->frame_tokens, (int64_t)p->B * p->H, p->q_st, gw * p->q_st,
                     (int64_t)p->frame_tokens * p->q_st, p->q_sh, p->bw, p->bh);
    ok = ok && encode_map5(&tm_kf, p->k_cache, p->d, gw, gh, p->H, p->n_pages, p->kv_st, gw * p->kv_st, p->kv_sh,
                           p->kv_sp, p->bw, p->bh, eb);
    ok = ok && encode_map5(&tm_vf, p->v_cache, p->d, gw, gh, p->H, p->n_pages, p->kv_st, gw * p->kv_st, p->kv_sh,
                           p->kv_sp, p->bw, p->bh, eb);
    tm_k8 = tm_kf;
    tm_v8 = tm_vf;
  } else {
    ok = encode_map(&tm_q, p->q, p->d, p->Lq, p->H, p->B, p->q_st, p->q_sh, p->q_sb, blk);
    ok = ok && encode_map(&tm_k8, p->k_cache, p->d, p->frame_tokens, p->H, p->n_pages, p->kv_st, p->kv_sh, p->kv_sp, 8, eb);
    ok = ok && encode_map(&tm_v8, p->v_cache, p->d, p->frame_tokens, p->H, p->n_pages, p->kv_st, p->kv_sh, p->kv_sp, 8, eb);
    ok = ok && encode_map(&tm_kf, p->k_cache, p->d, p->frame_tokens, p->H, p->n_pages, p->kv_st, p->kv_sh, p->kv_sp,
                          has_full ? half : 8, eb);
    ok = ok && encode_map(&tm_vf, p->v_cache, p->d, p->frame_tokens, p->H, p->n_pages, p->kv_st, p->kv_sh, p->kv_sp,
                          has_full ? half : 8, eb);
  }
  CUtensorMap tm_tk = tm_q, tm_tv = tm_q;      // placeholders when there is no text
  if (p->Lt > 0) {
    ok = ok && encode_map(&tm_tk, p->text_k, p->d, p->Lt, p->H, p->B, p->t_st, p->t_sh, p->t_sb, half);
    ok = ok && encode_map(&tm_tv, p->text_v, p->d, p->Lt, p->H, p->B, p->t_st, p->t_sh, p->t_sb, half);
  }
  if (!ok) return cuda_failed((int)cudaErrorUnknown);

  li::AttnParams ap;
  std::memset(&ap, 0, sizeof(ap));
  ap.tl = dv.tl;
  ap.B = p->B; ap.H = p->H; ap.Lq = p->Lq; ap.T_f = p->frame_tokens; ap.n_cur = p->n_cur_frames;
  ap.Nqb = dv.Nqb; ap.Nc = dv.Nc; ap.kmax = kmax; ap.has_box_full = has_full; ap.Lt = p->Lt;
  ap.no_split = (p->flags & LI_FLAG_NO_SPLIT) ? 1 : 0;
  if (p->flags & LI_FLAG_KV_FP8) { ap.k_scale = p->k_scale; ap.v_scale = p->v_scale; }
  const float scale = p->softmax_scale != 0.f ? p->softmax_scale : 1.0f / std::sqrt((float)p->d);
  ap.scale_log2 = scale * 1.4426950408889634f;
  ap.frame_idx = p->frame_idx; ap.sel_idx = sel_idx; ap.sel_cnt = sel_cnt;
  ap.o = (uint16_t *)o; ap.lse = lse_opt;
  if (have_ws) {
    ap.part_o = (float *)((char *)workspace + ws_bytes(p, dv));
    ap.part_ml = (float2 *)((char *)ap.part_o + ws_split_o_bytes(p));
  }
  int64_t n = 0;
  const int e = li::launch_attn(ap, dv.meta, p->d, blk, tm_q, tm_tk, tm_tv, tm_kf, tm_k8, tm_vf, tm_v8, (cudaStream_t)cuda_stream, &n);
  g_launches += n;
  return e == 0 ? LI_OK : cuda_failed(e);
}

int li_quantize_pages(const li_problem *p, const void *k_src, const void *v_src, const int32_t *pages_dev, int32_t n_list,
                      void *cuda_stream) {
  if (p == nullptr || !(p->flags & LI_FLAG_KV_FP8)) return LI_ERR_INVALID_ARG;
  if (p->H <= 0 || p->frame_tokens <= 0 || p->n_pages <= 0 || p->k_cache == nullptr || p->v_cache == nullptr ||
      p->k_scale == nullptr || p->v_scale == nullptr)
    return LI_ERR_INVALID_ARG;
  if (p->d != 128) return LI_ERR_UNSUPPORTED;
  if (n_list < 0 || (n_list > 0 && (k_src == nullptr || v_src == nullptr || pages_dev == nullptr))) return LI_ERR_INVALID_ARG;
  if ((((uintptr_t)k_src | (uintptr_t)v_src | (uintptr_t)p->k_cache | (uintptr_t)p->v_cache) & 15u) != 0) return LI_ERR_INVALID_ARG;
  if (p->kv_sp % 16 != 0 || p->kv_sh % 16 != 0 || p->kv_st % 16 != 0 || p->kv_st < p->d) return LI_ERR_INVALID_ARG;
  li::QuantParams qp;
  std::memset(&qp, 0, sizeof(qp));
  qp.H = p->H; qp.T_f = p->frame_tokens; qp.d = p->d; qp.n_pages = p->n_pages;
  qp.k_src = (const uint16_t *)k_src; qp.v_src = (const uint16_t *)v_src;
  qp.k_cache = (uint8_t *)const_cast<void *>(p->k_cache); qp.v_cache = (uint8_t *)const_cast<void *>(p->v_cache);
  qp.kv_sp = p->kv_sp; qp.kv_sh = p->kv_sh; qp.kv_st = p->kv_st;
  qp.k_scale = p->k_scale; qp.v_scale = p->v_scale; qp.pages = pages_dev;
  int64_t n = 0;
  const int e = li::launch_quantize_pages(qp, n_list, (cudaStream_t)cuda_stream, &n);
  g_launches += n;
  return e == 0 ? LI_OK : cuda_failed(e);
}

int li_validate(const li_problem *p, const int32_t *sel_idx, const int32_t *sel_cnt, int32_t kmax, int32_t *error_dev,
                void *cuda_stream) {
  Derived dv;
  int rc = check_problem(p, &dv);
  if (rc != LI_OK) return rc;
  if (error_dev == nullptr || ((sel_idx == nullptr) != (sel_cnt == nullptr)) || (sel_idx != nullptr && kmax < 1))
    return LI_ERR_INVALID_ARG;
  li::ValidateParams vp;
  std::memset(&vp, 0, sizeof(vp));
  vp.tl = dv.tl;
  vp.B = p->B; vp.H = p->H; vp.Nqb = dv.Nqb; vp.T_f = p->frame_tokens; vp.blk = p->block_k; vp.n_cur = p->n_cur_frames;
  vp.n_pages = p->n_pages; vp.kmax = kmax; vp.Mmax = dv.Mmax;
  vp.frame_idx = p->frame_idx; vp.sel_idx = sel_idx; vp.sel_cnt = sel_cnt; vp.err = error_dev;
  int64_t n = 0;
  const int e = li::launch_validate(vp, dv.meta, (cudaStream_t)cuda_stream, &n);
  g_launches += n;
  return e == 0 ? LI_OK : cuda_failed(e);
}

size_t li_policy_workspace_bytes(void) { return li::kPolicyWorkspaceBytes; }

int li_context_policy(const li_policy *pp, int32_t *frame_idx_out, int32_t frame_idx_capacity, li_policy_result *result_dev,
                      void *workspace, size_t workspace_bytes, void *cuda_stream) {
  if (pp == nullptr || frame_idx_out == nullptr || result_dev == nullptr) return LI_ERR_INVALID_ARG;
  if (pp->z_prev1 == nullptr || pp->z_prev2 == nullptr || pp->n_latent <= 0) return LI_ERR_INVALID_ARG;
  if (((uintptr_t)pp->z_prev1 & 15u) || ((uintptr_t)pp->z_prev2 & 15u)) return LI_ERR_INVALID_ARG;
  if (pp->latent_bf16 != 0 && pp->latent_bf16 != 1) return LI_ERR_INVALID_ARG;
  if (!(pp->alpha > 0.f && pp->alpha <= 1.f) || !(pp->kappa > 0.f) || pp->L_max < 1) return LI_ERR_INVALID_ARG;
  if (pp->ema_state == nullptr) return LI_ERR_INVALID_ARG;
  if (pp->n_cand < 0 || pp->n_mem < 0 || pp->n_win < 0 || pp->n_cur < 0) return LI_ERR_INVALID_ARG;
  if ((pp->n_cand > 0 && pp->s_pose == nullptr) || (pp->n_mem > 0 && pp->mem_pages == nullptr) ||
      (pp->n_win > 0 && pp->win_pages == nullptr) || (pp->n_cur > 0 && pp->cur_pages == nullptr))
    return LI_ERR_INVALID_ARG;
  const int64_t need = (int64_t)pp->n_mem + (pp->L_max < pp->n_win ? pp->L_max : pp->n_win) + pp->n_cur;
  if (frame_idx_capacity < need) return LI_ERR_INVALID_ARG;
  if (workspace == nullptr || workspace_bytes < li::kPolicyWorkspaceBytes || ((uintptr_t)workspace & 255u)) return LI_ERR_WORKSPACE;
  int64_t n = 0;
  const int e = li::launch_policy(*pp, frame_idx_out, result_dev, (double *)workspace, (cudaStream_t)cuda_stream, &n);
  g_launches += n;
  return e == 0 ? LI_OK : cuda_failed(e);
}

int64_t li_launch_count(void) { return g_launches.load(); }
void li_reset_launch_count(void) { g_launches.store(0); }

const char *li_strerror(int code) {
  switch (code) {
    case LI_OK: return "ok";
    case LI_ERR_INVALID_ARG: return "invalid argument";
    case LI_ERR_UNSUPPORTED: return "unsupported configuration";
    case LI_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case LI_ERR_CUDA: return "CUDA error";
    case LI_ERR_TOO_LARGE: return "problem needs more scratch than LI_STATIC_SCRATCH_BYTES (use li_block_select with a workspace)";
    default: return "unknown error";
  }
}

int li_version(void) { return LI_VERSION; }
int li_last_cuda_error(void) { return t_last_cuda_error; }

}  // extern "C"
