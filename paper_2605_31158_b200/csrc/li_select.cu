// li_select.cu -- li_block_select for sm_100a (Eq. 9-10).
//   kernel 1  li_pool_kernel       : block means of Q and of the historical K (K rows fetched through the
//                                    frame-index list, in place).  HBM-bound streaming reduction: every Q and
//                                    historical-K byte is read exactly once with 16-byte loads.
//   kernel 2  li_score_kernel      : scores qbar_i . kbar_m / sqrt(d) (fp32) -> order-preserving uint32 keys.
//   kernel 3  li_topk_kernel       : per-row top-k by an MSB-first radix select on the keys; ties -> lowest block
//                                    index; indices written ascending.
#include "li_internal.h"

namespace li {

// programmatic dependent launch: let the next kernel of the stream start its prologue early / wait for the
// previous kernel's results
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ uint4 ldg_stream(const void *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void add_bf16x8(float (&acc)[8], const uint4 &v) {
  acc[0] += __uint_as_float(v.x << 16);
  acc[1] += __uint_as_float(v.x & 0xffff0000u);
  acc[2] += __uint_as_float(v.y << 16);
  acc[3] += __uint_as_float(v.y & 0xffff0000u);
  acc[4] += __uint_as_float(v.z << 16);
  acc[5] += __uint_as_float(v.z & 0xffff0000u);
  acc[6] += __uint_as_float(v.w << 16);
  acc[7] += __uint_as_float(v.w & 0xffff0000u);
}

constexpr int kPoolThreads = 256;

// grid = (Nqb + Mmax, H, B).  blockIdx.x < Nqb: query block; otherwise historical K block m = x - Nqb.
template <int D, bool K3D>
__global__ void __launch_bounds__(kPoolThreads) li_pool_kernel(const SelectParams p, const BatchMeta meta) {
  constexpr int TPR = D / 8;                 // threads per row (16-byte loads)
  constexpr int RPP = kPoolThreads / TPR;    // rows per pass
  constexpr int kMaxIter = 128 / RPP;        // passes for the largest block (128 rows); bf16 zero adds nothing
  __shared__ float red[RPP][D];
  pdl_launch_dependents();
  const int h = blockIdx.y, b = blockIdx.z;
  const int r0 = threadIdx.x / TPR, cofs = (threadIdx.x % TPR) * 8;
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  int nvalid;
  float *out;
  int out_stride = 1;

  const Tiling tl = p.tl;
  // 3-D blocks: row r of block m = (tg, hb, wb) is frame tg*bt + r/32, grid row hb*bh + (r%32)/bw,
  // grid column wb*bw + (r%32)%bw; rows outside the grid or past the region's last frame are padding (not loaded,
  // not counted: "masked loads").  Returns the token's row inside its frame, or -1 for padding.
  auto row3d = [&](int m, int r, int n_reg, int &f) -> int {
    const int per = tl.Hb * tl.Wb, tg = m / per, rem = m - tg * per, hb = rem / tl.Wb, wb = rem - hb * tl.Wb;
    const int within = r & 31, hh = within / tl.bw, ww = within - hh * tl.bw;
    f = tg * tl.bt + (r >> 5);
    const int y = hb * tl.bh + hh;
    return (f < n_reg && y < tl.gh) ? y * tl.gw + wb * tl.bw + ww : -1;
  };
  auto count3d = [&](int m, int n_reg) -> int {
    const int per = tl.Hb * tl.Wb, tg = m / per, hb = (m - tg * per) / tl.Wb;
    return min(tl.bt, n_reg - tg * tl.bt) * min(tl.bh, tl.gh - hb * tl.bh) * tl.bw;
  };

  if ((int)blockIdx.x < p.Nqb) {
    const int i = blockIdx.x;
    uint4 v[kMaxIter];
    if constexpr (K3D) {
      const int n_reg = p.Lq / p.T_f;
      nvalid = count3d(i, n_reg);
      const uint16_t *base = p.q + b * p.q_sb + h * p.q_sh + cofs;
#pragma unroll
      for (int it = 0; it < kMaxIter; ++it) {
        const int r = r0 + it * RPP;
        int f;
        const int row = r < p.blk ? row3d(i, r, n_reg, f) : -1;
        v[it] = row >= 0 ? ldg_stream(base + ((int64_t)f * p.T_f + row) * p.q_st) : make_uint4(0, 0, 0, 0);
      }
    } else {
      const int t0 = i * p.blk;
      nvalid = min(p.blk, p.Lq - t0);
      const uint16_t *base = p.q + b * p.q_sb + h * p.q_sh + (int64_t)t0 * p.q_st + cofs;
#pragma unroll
      for (int it = 0; it < kMaxIter; ++it) {
        const int r = r0 + it * RPP;
        v[it] = r < nvalid ? ldg_stream(base + (int64_t)r * p.q_st) : make_uint4(0, 0, 0, 0);
      }
    }
#pragma unroll
    for (int it = 0; it < kMaxIter; ++it) add_bf16x8(acc, v[it]);
    out = p.qbar + (((int64_t)b * p.H + h) * p.Nqb + i) * D;
  } else {
    const int m = blockIdx.x - p.Nqb;
    const int foff = meta.frame_off[b];
    const int n_hist = meta.frame_off[b + 1] - foff - p.n_cur;
    if (m >= tl.num_blocks(n_hist, p.T_f, p.blk)) return;          // m >= M_b (whole CTA exits together)
    const uint16_t *base = p.k_cache + h * p.kv_sh + cofs;
    const int32_t *pages = p.frame_idx + foff;
    uint4 v[kMaxIter];
    if constexpr (K3D) {
      nvalid = count3d(m, n_hist);
      if (p.slice_cache != nullptr) {
        // page-resident patch sums (li_pool_pages): the block mean from <= bt cached rows, one channel per thread
        if (threadIdx.x < D) {
          const int per = tl.Hb * tl.Wb, tg = m / per, patch = m - tg * per;
          const int nf = min(tl.bt, n_hist - tg * tl.bt);
          float s = 0.f;
          for (int f = 0; f < nf; ++f)
            s += __ldg(p.slice_cache + (((int64_t)__ldg(pages + tg * tl.bt + f) * p.H + h) * per + patch) * D + threadIdx.x);
          p.kbar[(((int64_t)b * p.H + h) * D + threadIdx.x) * p.Mp + m] = s / (float)nvalid;
        }
        return;
      }
#pragma unroll
      for (int it = 0; it < kMaxIter; ++it) {
        const int r = r0 + it * RPP;
        int f;
        const int row = r < p.blk ? row3d(m, r, n_hist, f) : -1;
        v[it] = make_uint4(0, 0, 0, 0);
        if (row >= 0) v[it] = ldg_stream(base + __ldg(pages + f) * p.kv_sp + row * p.kv_st);
      }
    } else {
      const int L_hist = n_hist * p.T_f;
      const int t0 = m * p.blk;
      nvalid = min(p.blk, L_hist - t0);
#pragma unroll
      for (int it = 0; it < kMaxIter; ++it) {
        const int r = r0 + it * RPP;
        v[it] = make_uint4(0, 0, 0, 0);
        if (r < nvalid) {
          const int t = t0 + r;
          const int pg = t / p.T_f;
          const int row = t - pg * p.T_f;
          const int page = __ldg(pages + pg);
          v[it] = ldg_stream(base + page * p.kv_sp + row * p.kv_st);
        }
      }
    }
#pragma unroll
    for (int it = 0; it < kMaxIter; ++it) add_bf16x8(acc, v[it]);
    out = p.kbar + ((int64_t)b * p.H + h) * D * p.Mp + m;          // kbar is stored TRANSPOSED: [B,H,d,Mp]
    out_stride = p.Mp;
  }

#pragma unroll
  for (int e = 0; e < 8; ++e) red[r0][cofs + e] = acc[e];
  __syncthreads();
  if (threadIdx.x < D) {
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < RPP; ++r) s += red[r][threadIdx.x];
    out[(int64_t)threadIdx.x * out_stride] = s / (float)nvalid;    // Eq. 9: true cardinality |Q_i|, |K_m|
  }
}

constexpr int kRowsPerWarp = 8;              // query-block rows scored together by one warp
constexpr int kKeysPerLane = 16;             // top-k register fast path covers M <= 512 historical blocks
constexpr int kTopkWarps = 8;                // rows (warps) per CTA of the top-k kernel

__device__ __forceinline__ uint32_t order_key(float s) {
  const uint32_t u = __float_as_uint(s);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);   // unsigned order == float order
}

// Scores (Eq. 10).  grid = (ceil(Mmax/32), ceil(Nqb/8), B*H), 4 warps per CTA.  The work is latency-bound (a few MFLOP
// spread over thousands of CTAs), so the dependent chain of every warp is kept short: lane = one historical block m,
// warp w walks channels [w*D/4, (w+1)*D/4) of its pooled key row (one coalesced 128-byte line per channel, kbar is
// channel-major) against 8 pooled query rows broadcast from shared memory = 8 independent fp32 FMA chains; the 4
// partial sums of a score are added in a fixed order (w = 0..3) through shared memory.  Output: order-preserving keys
// [B,H,Nqb,Mmax] (+ scores).
constexpr int kScoreWarps = 4;
template <int D>
__global__ void __launch_bounds__(kScoreWarps * 32) li_score_kernel(const SelectParams p, const BatchMeta meta) {
  __shared__ __align__(16) float sq[kRowsPerWarp * D];
  __shared__ float part[kScoreWarps][kRowsPerWarp][32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int bh = blockIdx.z, b = bh / p.H;
  const int i0 = blockIdx.y * kRowsPerWarp;
  const int n_hist = meta.frame_off[b + 1] - meta.frame_off[b] - p.n_cur;
  const int M = p.tl.num_blocks(n_hist, p.T_f, p.blk);
  const int m = blockIdx.x * 32 + lane;
  if ((int)blockIdx.x * 32 >= M) return;
  pdl_launch_dependents();
  pdl_wait();                                              // qbar / kbar come from li_pool_kernel

  // kbar is [B,H,d,Mp] (written transposed by the pool kernel): for a fixed channel the 32 lanes read 32
  // consecutive floats = one 128-byte line.  Lanes past M read padding and their results are dropped.
  constexpr int DW = D / kScoreWarps;                        // channels per warp
  const float *kT = p.kbar + ((int64_t)bh * D + warp * DW) * p.Mp + m;
  float kv[DW];
#pragma unroll
  for (int c = 0; c < DW; ++c) kv[c] = __ldg(kT + (int64_t)c * p.Mp);   // all in flight while the q rows are staged
  for (int t = threadIdx.x; t < kRowsPerWarp * D / 4; t += kScoreWarps * 32) {
    const int g = t / (D / 4);
    reinterpret_cast<float4 *>(sq)[t] =
        (i0 + g < p.Nqb) ? __ldg(reinterpret_cast<const float4 *>(p.qbar + ((int64_t)bh * p.Nqb + i0) * D) + t)
                         : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();

  float acc[kRowsPerWarp];
#pragma unroll
  for (int g = 0; g < kRowsPerWarp; ++g) acc[g] = 0.f;
#pragma unroll
  for (int c = 0; c < DW; c += 4) {
#pragma unroll
    for (int g = 0; g < kRowsPerWarp; ++g) {
      const float4 qv = *reinterpret_cast<const float4 *>(sq + g * D + warp * DW + c);
      acc[g] = fmaf(qv.x, kv[c], acc[g]);
      acc[g] = fmaf(qv.y, kv[c + 1], acc[g]);
      acc[g] = fmaf(qv.z, kv[c + 2], acc[g]);
      acc[g] = fmaf(qv.w, kv[c + 3], acc[g]);
    }
  }
#pragma unroll
  for (int g = 0; g < kRowsPerWarp; ++g) part[warp][g][lane] = acc[g];
  __syncthreads();
  if (m < M) {
#pragma unroll
    for (int gg = 0; gg < kRowsPerWarp / kScoreWarps; ++gg) {     // warp w finishes rows w*2, w*2+1
      const int g = warp * (kRowsPerWarp / kScoreWarps) + gg;
      if (i0 + g < p.Nqb) {
        const float dot = ((part[0][g][lane] + part[1][g][lane]) + part[2][g][lane]) + part[3][g][lane];
        const float sc = dot * p.inv_sqrt_d + 0.0f;          // -0 -> +0 so that equal scores have equal keys
        p.keys[((int64_t)bh * p.Nqb + i0 + g) * p.Mmax + m] = order_key(sc);
        if (p.scores != nullptr) p.scores[((int64_t)bh * p.Nqb + i0 + g) * p.score_pitch + m] = sc;
      }
    }
  }
}

// Top_k (Eq. 10).  One warp per (call, head, query block) row; grid = ceil(B*H*Nqb / 8) CTAs of 8 warps.
// MSB-first radix select of the k-th largest key, then one ordered pass that emits, ascending, every block above
// the threshold plus the lowest-index blocks equal to it.
__global__ void __launch_bounds__(kTopkWarps * 32) li_topk_kernel(const SelectParams p, const BatchMeta meta) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * kTopkWarps + warp;
  if (row >= (int64_t)p.B * p.H * p.Nqb) return;
  pdl_launch_dependents();
  pdl_wait();                                              // keys come from li_score_kernel
  const int b = (int)(row / ((int64_t)p.H * p.Nqb));
  const int n_hist = meta.frame_off[b + 1] - meta.frame_off[b] - p.n_cur;
  const int M = p.tl.num_blocks(n_hist, p.T_f, p.blk);
  const int k = min(meta.top_k[b], M);
  const uint32_t *key = p.keys + row * p.Mmax;
  int32_t *out = p.sel_idx + row * p.kmax;
  if (lane == 0) p.sel_cnt[row] = k;
  if (k > 0) {
    // T = k-th largest key: build it MSB first, keeping count(key >= T) >= k
    uint32_t T = 0;
    int c_gt = 0;
    if (M <= 32 * kKeysPerLane) {
      // fast path: each lane keeps its keys (block m = lane + 32*x) in registers; absent blocks get key 0,
      // which is below every real key (order_key never returns 0 for a non-NaN score)
      uint32_t kr[kKeysPerLane];
#pragma unroll
      for (int x = 0; x < kKeysPerLane; ++x) kr[x] = (lane + 32 * x < M) ? key[lane + 32 * x] : 0u;
      for (int bit = 31; bit >= 0; --bit) {
        const uint32_t cand = T | (1u << bit);
        int c = 0;
#pragma unroll
        for (int x = 0; x < kKeysPerLane; ++x) c += kr[x] >= cand;
        c = __reduce_add_sync(0xffffffffu, c);
        if (c >= k) T = cand;
      }
#pragma unroll
      for (int x = 0; x < kKeysPerLane; ++x) c_gt += kr[x] > T;
      c_gt = __reduce_add_sync(0xffffffffu, c_gt);
      int need_eq = k - c_gt;                                // ties at the threshold: lowest index first
      int pos = 0;
#pragma unroll
      for (int x = 0; x < kKeysPerLane; ++x) {
        const bool gt = kr[x] > T;
        const bool eq = kr[x] == T && T != 0u;
        const uint32_t eq_mask = __ballot_sync(0xffffffffu, eq);
        const uint32_t lt = (1u << lane) - 1u;
        const bool take = gt || (eq && __popc(eq_mask & lt) < need_eq);
        const uint32_t take_mask = __ballot_sync(0xffffffffu, take);
        if (take) out[pos + __popc(take_mask & lt)] = lane + 32 * x;
        pos += __popc(take_mask);
        need_eq -= min(need_eq, __popc(eq_mask));
      }
    } else {
      for (int bit = 31; bit >= 0; --bit) {
        const uint32_t cand = T | (1u << bit);
        int c = 0;
        for (int m = lane; m < M; m += 32) c += key[m] >= cand;
        c = __reduce_add_sync(0xffffffffu, c);
        if (c >= k) T = cand;
      }
      for (int m = lane; m < M; m += 32) c_gt += key[m] > T;
      c_gt = __reduce_add_sync(0xffffffffu, c_gt);
      int need_eq = k - c_gt;
      int pos = 0;
      for (int m0 = 0; m0 < M; m0 += 32) {
        const int m = m0 + lane;
        const uint32_t kv = m < M ? key[m] : 0u;
        const bool gt = m < M && kv > T;
        const bool eq = m < M && kv == T;
        const uint32_t eq_mask = __ballot_sync(0xffffffffu, eq);
        const uint32_t lt = (1u << lane) - 1u;
        const bool take = gt || (eq && __popc(eq_mask & lt) < need_eq);
        const uint32_t take_mask = __ballot_sync(0xffffffffu, take);
        if (take) out[pos + __popc(take_mask & lt)] = m;
        pos += __popc(take_mask);
        need_eq -= min(need_eq, __popc(eq_mask));
      }
    }
  }
  for (int t = k + lane; t < p.kmax; t += 32) out[t] = -1;
}

// ----------------------------------------------------------------------------- page-resident pooled slices
// 3-D tiling only.  A 3-D block is bt frames x one bh x bw patch, and a frame's patch sum does not depend on
// where the frame sits in a call's logical list, so it is computed ONCE when the page is written:
//   cache [n_pages][H][Hb*Wb][D] fp32 = sum of the K rows of that frame's patch (rows inside the grid only).
// Selection then pools a historical block from <= bt cached rows instead of 128 K rows (1/32 of the bytes).
template <int D>
__global__ void __launch_bounds__(128) li_pool_pages_kernel(const SelectParams p, const int32_t *pages, float *cache) {
  constexpr int TPR = D / 8;                 // threads per row (16-byte loads)
  constexpr int RPP = 128 / TPR;             // rows per pass
  __shared__ float red[RPP][D];
  const Tiling tl = p.tl;
  const int patch = blockIdx.x, h = blockIdx.y, page = pages[blockIdx.z];
  const int hb = patch / tl.Wb, wb = patch - hb * tl.Wb;
  const int r0 = threadIdx.x / TPR, cofs = (threadIdx.x % TPR) * 8;
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  const uint16_t *base = p.k_cache + (int64_t)page * p.kv_sp + h * p.kv_sh + cofs;
#pragma unroll
  for (int it = 0; it < 32 / RPP; ++it) {
    const int r = r0 + it * RPP, hh = r / tl.bw, ww = r - hh * tl.bw, y = hb * tl.bh + hh;
    if (y < tl.gh) add_bf16x8(acc, ldg_stream(base + (int64_t)(y * tl.gw + wb * tl.bw + ww) * p.kv_st));
  }
#pragma unroll
  for (int e = 0; e < 8; ++e) red[r0][cofs + e] = acc[e];
  __syncthreads();
  if (threadIdx.x < D) {
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < RPP; ++r) s += red[r][threadIdx.x];
    cache[(((int64_t)page * p.H + h) * (tl.Hb * tl.Wb) + patch) * D + threadIdx.x] = s;
  }
}

int launch_pool_pages(const SelectParams &sp, const int32_t *pages, int n_list, float *cache, cudaStream_t st, int64_t *n_launches) {
  if (n_list <= 0) return 0;
  dim3 grid(sp.tl.Hb * sp.tl.Wb, sp.H, n_list);
  if (sp.d == 128) li_pool_pages_kernel<128><<<grid, 128, 0, st>>>(sp, pages, cache);
  else li_pool_pages_kernel<64><<<grid, 128, 0, st>>>(sp, pages, cache);
  if (n_launches) *n_launches += 1;
  return (int)cudaGetLastError();
}

int launch_select(const SelectParams &sp, const BatchMeta &meta, cudaStream_t st, int64_t *n_launches) {
  {
    dim3 grid(sp.Nqb + (sp.skip_k ? 0 : sp.Mmax), sp.H, sp.B);
    if (sp.tl.bt > 0) {
      if (sp.d == 128) li_pool_kernel<128, true><<<grid, kPoolThreads, 0, st>>>(sp, meta);
      else li_pool_kernel<64, true><<<grid, kPoolThreads, 0, st>>>(sp, meta);
    } else {
      if (sp.d == 128) li_pool_kernel<128, false><<<grid, kPoolThreads, 0, st>>>(sp, meta);
      else li_pool_kernel<64, false><<<grid, kPoolThreads, 0, st>>>(sp, meta);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return (int)e;
    if (n_launches) *n_launches += 1;
  }
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  if (sp.Mmax > 0) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((sp.Mmax + 31) / 32, (sp.Nqb + kRowsPerWarp - 1) / kRowsPerWarp, sp.B * sp.H);
    cfg.blockDim = dim3(kScoreWarps * 32);
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = sp.d == 128 ? cudaLaunchKernelEx(&cfg, li_score_kernel<128>, sp, meta)
                                : cudaLaunchKernelEx(&cfg, li_score_kernel<64>, sp, meta);
    if (e != cudaSuccess) return (int)e;
    if (n_launches) *n_launches += 1;
  }
  {
    const int64_t rows = (int64_t)sp.B * sp.H * sp.Nqb;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((rows + kTopkWarps - 1) / kTopkWarps));
    cfg.blockDim = dim3(kTopkWarps * 32);
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, li_topk_kernel, sp, meta);
    if (e != cudaSuccess) return (int)e;
    if (n_launches) *n_launches += 1;
  }
  return 0;
}

}  // namespace li
