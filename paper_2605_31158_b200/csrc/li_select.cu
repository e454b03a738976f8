// li_select.cu -- li_block_select for sm_100a (Eq. 9-10).
//   kernel 1  li_pool_kernel       : block means of Q and of the historical K (K rows fetched through the
//                                    frame-index list, in place).  HBM-bound streaming reduction: every Q and
//                                    historical-K byte is read exactly once with 16-byte loads.
//   kernel 2  li_score_topk_kernel : scores qbar_i . kbar_m / sqrt(d) (fp32) and the per-row top-k by an
//                                    MSB-first radix select on order-preserving keys; ties -> lowest block index;
//                                    indices written ascending.
#include "li_internal.h"

namespace li {

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
template <int D>
__global__ void __launch_bounds__(kPoolThreads) li_pool_kernel(const SelectParams p, const BatchMeta meta) {
  constexpr int TPR = D / 8;                 // threads per row (16-byte loads)
  constexpr int RPP = kPoolThreads / TPR;    // rows per pass
  constexpr int kMaxIter = 128 / RPP;        // passes for the largest block (128 rows); bf16 zero adds nothing
  __shared__ float red[RPP][D];
  const int h = blockIdx.y, b = blockIdx.z;
  const int r0 = threadIdx.x / TPR, cofs = (threadIdx.x % TPR) * 8;
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  int nvalid;
  float *out;

  if ((int)blockIdx.x < p.Nqb) {
    const int i = blockIdx.x;
    const int t0 = i * p.blk;
    nvalid = min(p.blk, p.Lq - t0);
    const uint16_t *base = p.q + b * p.q_sb + h * p.q_sh + (int64_t)t0 * p.q_st + cofs;
    uint4 v[kMaxIter];
#pragma unroll
    for (int it = 0; it < kMaxIter; ++it) {
      const int r = r0 + it * RPP;
      v[it] = r < nvalid ? ldg_stream(base + (int64_t)r * p.q_st) : make_uint4(0, 0, 0, 0);
    }
#pragma unroll
    for (int it = 0; it < kMaxIter; ++it) add_bf16x8(acc, v[it]);
    out = p.qbar + (((int64_t)b * p.H + h) * p.Nqb + i) * D;
  } else {
    const int m = blockIdx.x - p.Nqb;
    const int foff = meta.frame_off[b];
    const int n_hist = meta.frame_off[b + 1] - foff - p.n_cur;
    const int L_hist = n_hist * p.T_f;
    const int t0 = m * p.blk;
    if (t0 >= L_hist) return;                // m >= M_b (whole CTA exits together)
    nvalid = min(p.blk, L_hist - t0);
    const uint16_t *base = p.k_cache + h * p.kv_sh + cofs;
    const int32_t *pages = p.frame_idx + foff;
    uint4 v[kMaxIter];
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
#pragma unroll
    for (int it = 0; it < kMaxIter; ++it) add_bf16x8(acc, v[it]);
    out = p.kbar + (((int64_t)b * p.H + h) * p.Mmax + m) * D;
  }

#pragma unroll
  for (int e = 0; e < 8; ++e) red[r0][cofs + e] = acc[e];
  __syncthreads();
  if (threadIdx.x < D) {
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < RPP; ++r) s += red[r][threadIdx.x];
    out[threadIdx.x] = s / (float)nvalid;    // Eq. 9: true cardinality |Q_i|, |K_m|
  }
}

constexpr int kRowsPerCta = 8;               // query-block rows per CTA == warps per CTA

__device__ __forceinline__ uint32_t order_key(float s) {
  const uint32_t u = __float_as_uint(s);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);   // unsigned order == float order
}

// grid = (ceil(Nqb / 8), H, B), 256 threads, dynamic smem = 8 * Mmax * 4 bytes (keys) + 8 * D * 4 (qbar rows)
template <int D>
__global__ void __launch_bounds__(kRowsPerCta * 32) li_score_topk_kernel(const SelectParams p, const BatchMeta meta) {
  extern __shared__ uint32_t sm[];
  float *sq = reinterpret_cast<float *>(sm);                 // [8][D]
  uint32_t *skey = sm + kRowsPerCta * D;                     // [8][Mmax]
  const int h = blockIdx.y, b = blockIdx.z;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i0 = blockIdx.x * kRowsPerCta;
  const int n_hist = meta.frame_off[b + 1] - meta.frame_off[b] - p.n_cur;
  const int M = (n_hist * p.T_f + p.blk - 1) / p.blk;
  const int k = min(meta.top_k[b], M);
  const int64_t bh = (int64_t)b * p.H + h;

  for (int t = threadIdx.x; t < kRowsPerCta * D; t += blockDim.x) {
    const int g = t / D, c = t % D;
    sq[t] = (i0 + g < p.Nqb) ? p.qbar[(bh * p.Nqb + i0 + g) * D + c] : 0.f;
  }
  __syncthreads();

  // ---- scores (Eq. 10): a warp takes 4 historical blocks at a time, lanes across d; the 4 x 8 partial dot
  // products per lane are summed over the 32 lanes by a transposing butterfly (31 shuffles instead of 160),
  // after which lane (mm*8 + g) holds the finished score of block m0+mm for query row g ----
  constexpr int EPL = D / 32;                                // elements per lane (4 or 2)
  float qreg[kRowsPerCta][EPL];
#pragma unroll
  for (int g = 0; g < kRowsPerCta; ++g)
#pragma unroll
    for (int e = 0; e < EPL; ++e) qreg[g][e] = sq[g * D + lane * EPL + e];
  for (int m0 = warp * 4; m0 < M; m0 += kRowsPerCta * 4) {
    float kv[4][EPL];
#pragma unroll
    for (int mm = 0; mm < 4; ++mm) {
      const int m = min(m0 + mm, M - 1);
      const float *kr = p.kbar + (bh * p.Mmax + m) * D + lane * EPL;
      if constexpr (EPL == 4) {
        const float4 t = *reinterpret_cast<const float4 *>(kr);
        kv[mm][0] = t.x; kv[mm][1] = t.y; kv[mm][2] = t.z; kv[mm][3] = t.w;
      } else {
        const float2 t = *reinterpret_cast<const float2 *>(kr);
        kv[mm][0] = t.x; kv[mm][1] = t.y;
      }
    }
    float v[32];
#pragma unroll
    for (int mm = 0; mm < 4; ++mm)
#pragma unroll
      for (int g = 0; g < kRowsPerCta; ++g) {
        float a = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) a = fmaf(qreg[g][e], kv[mm][e], a);
        v[mm * 8 + g] = a;
      }
#pragma unroll
    for (int w = 16; w >= 1; w >>= 1) {
      const bool up = (lane & w) != 0;                       // this lane keeps the upper half of the values
#pragma unroll
      for (int x = 0; x < w; ++x) {
        const float keep = up ? v[x + w] : v[x];
        const float send = up ? v[x] : v[x + w];
        v[x] = keep + __shfl_xor_sync(0xffffffffu, send, w);
      }
    }
    const int m = m0 + (lane >> 3), g = lane & 7;
    if (m < M && i0 + g < p.Nqb) {
      const float sc = v[0] * p.inv_sqrt_d + 0.0f;           // -0 -> +0 so that equal scores have equal keys
      skey[g * p.Mmax + m] = order_key(sc);
      if (p.scores != nullptr) p.scores[(bh * p.Nqb + i0 + g) * p.score_pitch + m] = sc;
    }
  }
  __syncthreads();

  // ---- Top_k (Eq. 10): warp per query-block row ----
  const int i = i0 + warp;
  if (i >= p.Nqb) return;
  const uint32_t *key = skey + warp * p.Mmax;
  int32_t *out = p.sel_idx + (bh * p.Nqb + i) * p.kmax;
  if (lane == 0) p.sel_cnt[bh * p.Nqb + i] = k;
  if (k > 0) {
    // T = k-th largest key: build it MSB first, keeping count(key >= T) >= k
    uint32_t T = 0;
    for (int bit = 31; bit >= 0; --bit) {
      const uint32_t cand = T | (1u << bit);
      int c = 0;
      for (int m = lane; m < M; m += 32) c += key[m] >= cand;
      c = __reduce_add_sync(0xffffffffu, c);
      if (c >= k) T = cand;
    }
    int c_gt = 0;
    for (int m = lane; m < M; m += 32) c_gt += key[m] > T;
    c_gt = __reduce_add_sync(0xffffffffu, c_gt);
    int need_eq = k - c_gt;                                  // ties at the threshold: lowest index first
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
  for (int t = k + lane; t < p.kmax; t += 32) out[t] = -1;
}

int launch_select(const SelectParams &sp, const BatchMeta &meta, cudaStream_t st, int64_t *n_launches) {
  {
    dim3 grid(sp.Nqb + sp.Mmax, sp.H, sp.B);
    if (sp.d == 128) li_pool_kernel<128><<<grid, kPoolThreads, 0, st>>>(sp, meta);
    else li_pool_kernel<64><<<grid, kPoolThreads, 0, st>>>(sp, meta);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return (int)e;
    if (n_launches) *n_launches += 1;
  }
  {
    dim3 grid((sp.Nqb + kRowsPerCta - 1) / kRowsPerCta, sp.H, sp.B);
    const size_t smem = (size_t)kRowsPerCta * (sp.Mmax > 0 ? sp.Mmax : 1) * 4 + (size_t)kRowsPerCta * sp.d * 4;
    cudaError_t e;
    if (sp.d == 128) {
      e = cudaFuncSetAttribute(li_score_topk_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e != cudaSuccess) return (int)e;
      li_score_topk_kernel<128><<<grid, kRowsPerCta * 32, smem, st>>>(sp, meta);
    } else {
      e = cudaFuncSetAttribute(li_score_topk_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e != cudaSuccess) return (int)e;
      li_score_topk_kernel<64><<<grid, kRowsPerCta * 32, smem, st>>>(sp, meta);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return (int)e;
    if (n_launches) *n_launches += 1;
  }
  return 0;
}

}  // namespace li
