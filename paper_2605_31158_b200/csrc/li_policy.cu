// li_policy.cu -- li_context_policy for sm_100a: adaptive context management (Eq. 1-4) and the frame list
// memory | temporal window | current chunk that li_block_select / li_sparse_attn consume (include/li.h).
//
//   li_mse_partial_kernel   : Eq. 1, streaming reduction over the two latents (HBM-bound: 2 * n_latent * sizeof(elem)
//                             bytes, 16-byte loads, fp32 squared differences, fp64 sums; one partial per CTA, no atomics ->
//                             deterministic)
//   li_policy_finalize_kernel: one CTA: fixed-order fp64 sum of the partials, Eq. 2-4 in fp32 with explicitly rounded
//                             operations (the window length is an integer decided by floating point: the operation order
//                             is part of the interface, li.h), then the frame list and the result record.
#include <cuda_bf16.h>

#include "li_internal.h"

namespace li {

constexpr int kMseThreads = 256;
constexpr int kMseMaxCtas = 1024;

__device__ __forceinline__ uint4 ldg_stream16(const void *p) {
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}

__device__ __forceinline__ float sqdiff_bf16x2(uint32_t a, uint32_t b) {
  const float a0 = __uint_as_float(a << 16), a1 = __uint_as_float(a & 0xffff0000u);
  const float b0 = __uint_as_float(b << 16), b1 = __uint_as_float(b & 0xffff0000u);
  const float d0 = a0 - b0, d1 = a1 - b1;
  return fmaf(d0, d0, d1 * d1);
}

template <bool BF16>
__global__ void __launch_bounds__(kMseThreads) li_mse_partial_kernel(const void *za, const void *zb, int64_t n, double *partial) {
  constexpr int EPV = BF16 ? 8 : 4;                      // elements per 16-byte vector
  const int64_t n_vec = n / EPV;
  const int64_t stride = (int64_t)gridDim.x * kMseThreads;
  double acc = 0.0;
  auto sq = [](const uint4 &a, const uint4 &b) -> float {
    if (BF16) return (sqdiff_bf16x2(a.x, b.x) + sqdiff_bf16x2(a.y, b.y)) + (sqdiff_bf16x2(a.z, b.z) + sqdiff_bf16x2(a.w, b.w));
    const float d0 = __uint_as_float(a.x) - __uint_as_float(b.x), d1 = __uint_as_float(a.y) - __uint_as_float(b.y);
    const float d2 = __uint_as_float(a.z) - __uint_as_float(b.z), d3 = __uint_as_float(a.w) - __uint_as_float(b.w);
    return fmaf(d0, d0, d1 * d1) + fmaf(d2, d2, d3 * d3);
  };
  int64_t v = (int64_t)blockIdx.x * kMseThreads + threadIdx.x;
  for (; v + 3 * stride < n_vec; v += 4 * stride) {       // 8 independent 16-byte loads in flight per thread
    uint4 a[4], b[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      a[u] = ldg_stream16((const char *)za + (v + u * stride) * 16);
      b[u] = ldg_stream16((const char *)zb + (v + u * stride) * 16);
    }
    acc += (double)((sq(a[0], b[0]) + sq(a[1], b[1])) + (sq(a[2], b[2]) + sq(a[3], b[3])));   // one fp64 add per 4 vectors
  }
  for (; v < n_vec; v += stride) acc += (double)sq(ldg_stream16((const char *)za + v * 16), ldg_stream16((const char *)zb + v * 16));
  if (blockIdx.x == 0 && threadIdx.x < n - n_vec * EPV) {   // ragged tail: fewer than EPV elements
    const int64_t e = n_vec * EPV + threadIdx.x;
    float d;
    if (BF16) {
      const uint16_t *pa = (const uint16_t *)za, *pb = (const uint16_t *)zb;
      d = __uint_as_float((uint32_t)pa[e] << 16) - __uint_as_float((uint32_t)pb[e] << 16);
    } else {
      d = ((const float *)za)[e] - ((const float *)zb)[e];
    }
    acc += (double)(d * d);
  }
  // block reduction in a fixed order: warp shuffles, then warp 0 over the 8 warp sums
  __shared__ double wsum[kMseThreads / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < kMseThreads / 32; ++w) t += wsum[w];
    partial[blockIdx.x] = t;
  }
}

struct PolicyParams {
  li_policy pp;
  int32_t n_partial;
  const double *partial;
  int32_t *frame_idx_out;
  li_policy_result *result;
};

__global__ void __launch_bounds__(256) li_policy_finalize_kernel(const PolicyParams q) {
  asm volatile("griddepcontrol.wait;" ::: "memory");      // the partial sums come from li_mse_partial_kernel (PDL)
  const li_policy &pp = q.pp;
  __shared__ double dsum[8];
  __shared__ float smax[8];
  __shared__ int s_keep, s_L;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // Eq. 1: fixed-order sum of the per-CTA partials
  double acc = 0.0;
  for (int k = threadIdx.x; k < q.n_partial; k += 256) acc += q.partial[k];
  // Eq. 4: max_j S_pose(t, j)
  float mx = __int_as_float(0xff800000);
  for (int k = threadIdx.x; k < pp.n_cand; k += 256) mx = fmaxf(mx, pp.s_pose[k]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    acc += __shfl_down_sync(0xffffffffu, acc, o);
    mx = fmaxf(mx, __shfl_down_sync(0xffffffffu, mx, o));
  }
  if (lane == 0) { dsum[warp] = acc; smax[warp] = mx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    float m = smax[0];
    for (int w = 0; w < 8; ++w) { t += dsum[w]; m = fmaxf(m, smax[w]); }
    const float D_t = (float)(t / (double)pp.n_latent);
    // Eq. 2 (fp32, each operation rounded once)
    const bool valid = pp.ema_state[1] != 0.0f;
    const float D_bar = valid ? __fadd_rn(__fmul_rn(pp.alpha, D_t), __fmul_rn(__fsub_rn(1.0f, pp.alpha), pp.ema_state[0])) : D_t;
    pp.ema_state[0] = D_bar;
    pp.ema_state[1] = 1.0f;
    // Eq. 3: (L_max * kappa) / (Dbar + kappa), floor or nearest-even, clip to [1, L_max]
    const float x = __fdiv_rn(__fmul_rn((float)pp.L_max, pp.kappa), __fadd_rn(D_bar, pp.kappa));
    const float r = pp.round_nearest ? rintf(x) : floorf(x);
    const int L_t = (int)fminf(fmaxf(r, 1.0f), (float)pp.L_max);
    // Eq. 4: discard the retrieved memory iff max < tau (strict); nothing to keep without candidates
    const int keep = (pp.n_cand > 0 && !(m < pp.tau_pose)) ? 1 : 0;
    s_keep = keep;
    s_L = L_t;
    const int n_win_used = min(L_t, pp.n_win), n_hist = (keep ? pp.n_mem : 0) + n_win_used;
    q.result->D_t = D_t;
    q.result->D_bar = D_bar;
    q.result->L_t = L_t;
    q.result->keep_memory = keep;
    q.result->n_hist_frames = n_hist;
    q.result->n_frames = n_hist + pp.n_cur;
  }
  __syncthreads();
  // frame list: memory (if kept) | last min(L_t, n_win) window pages | current chunk
  const int n_mem = s_keep ? pp.n_mem : 0, n_win_used = min(s_L, pp.n_win);
  for (int k = threadIdx.x; k < n_mem; k += 256) q.frame_idx_out[k] = pp.mem_pages[k];
  for (int k = threadIdx.x; k < n_win_used; k += 256) q.frame_idx_out[n_mem + k] = pp.win_pages[pp.n_win - n_win_used + k];
  for (int k = threadIdx.x; k < pp.n_cur; k += 256) q.frame_idx_out[n_mem + n_win_used + k] = pp.cur_pages[k];
}

int launch_policy(const li_policy &pp, int32_t *frame_idx_out, li_policy_result *result, double *partial, cudaStream_t st,
                  int64_t *n_launches) {
  const int epv = pp.latent_bf16 ? 8 : 4;
  const int64_t n_vec = pp.n_latent / epv;
  int64_t g = (n_vec + (int64_t)kMseThreads * 4 - 1) / ((int64_t)kMseThreads * 4);   // >= 4 vectors per thread when large
  if (g < 1) g = 1;
  if (g > kMseMaxCtas) g = kMseMaxCtas;
  if (pp.latent_bf16) li_mse_partial_kernel<true><<<(int)g, kMseThreads, 0, st>>>(pp.z_prev1, pp.z_prev2, pp.n_latent, partial);
  else li_mse_partial_kernel<false><<<(int)g, kMseThreads, 0, st>>>(pp.z_prev1, pp.z_prev2, pp.n_latent, partial);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return (int)e;
  PolicyParams q;
  q.pp = pp;
  q.n_partial = (int)g;
  q.partial = partial;
  q.frame_idx_out = frame_idx_out;
  q.result = result;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(1);
  cfg.blockDim = dim3(256);
  cfg.stream = st;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  e = cudaLaunchKernelEx(&cfg, li_policy_finalize_kernel, q);
  if (e != cudaSuccess) return (int)e;
  if (n_launches) *n_launches += 2;
  return (int)cudaGetLastError();
}

}  // namespace li
