// li_fp8.cu -- FP8 (E4M3) K/V pages (include/li.h LI_FLAG_KV_FP8):
//   li_quantize_pages_kernel : quantise-on-write, bf16 rows -> e4m3 codes, one fp32 scale per head (HBM-bound: 4 bytes
//                              read + 2 written per element pair of K and V)
//   li_pool_k8_kernel        : Eq. 9 for the historical K blocks read from e4m3 pages: half the bytes of
//                              the bf16 pooling, same one-CTA-per-block streaming reduction
#include "li_internal.h"
#include "li_ptx.cuh"

namespace li {

__device__ __forceinline__ uint4 ldg_stream16(const void *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
// two fp32 -> two e4m3 codes (round to nearest even, saturating at +-448): lo in bits [0,8), hi in bits [8,16)
__device__ __forceinline__ uint32_t cvt_e4m3x2(float lo, float hi) {
  uint16_t r;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(hi), "f"(lo));
  return r;
}
// two e4m3 codes (low 16 bits) -> two fp32, exactly
__device__ __forceinline__ void e4m3x2_to_f32(uint32_t v, float &lo, float &hi) {
  uint32_t h2;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"((uint16_t)v));
  asm("{.reg .b16 a, b; mov.b32 {a, b}, %2; cvt.f32.f16 %0, a; cvt.f32.f16 %1, b;}" : "=f"(lo), "=f"(hi) : "r"(h2));
}

// grid = (ceil(H*T_f*d / (256*16)), n_list, 2 {K, V}); a thread converts 16 consecutive channels (32 B in, 16 B out)
__global__ void __launch_bounds__(256) li_quantize_pages_kernel(const QuantParams q) {
  const int page = q.pages[blockIdx.y];
  if ((unsigned)page >= (unsigned)q.n_pages) return;
  const bool is_v = blockIdx.z != 0;
  const int64_t per_page = (int64_t)q.H * q.T_f * q.d;
  const int64_t e0 = ((int64_t)blockIdx.x * 256 + threadIdx.x) * 16;   // first element of this thread inside the page
  if (e0 >= per_page) return;
  const int c = (int)(e0 % q.d);
  const int64_t row = e0 / q.d;
  const int t = (int)(row % q.T_f), h = (int)(row / q.T_f);
  const uint16_t *src = (is_v ? q.v_src : q.k_src) + (int64_t)blockIdx.y * per_page + e0;
  const float s = __ldg((is_v ? q.v_scale : q.k_scale) + h);
  const uint4 a = ldg_stream16(src), b = ldg_stream16(src + 8);
  const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
  uint32_t out[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float x0 = __fdiv_rn(__uint_as_float(w[2 * i] << 16), s), x1 = __fdiv_rn(__uint_as_float(w[2 * i] & 0xffff0000u), s);
    const float x2 = __fdiv_rn(__uint_as_float(w[2 * i + 1] << 16), s), x3 = __fdiv_rn(__uint_as_float(w[2 * i + 1] & 0xffff0000u), s);
    out[i] = cvt_e4m3x2(x0, x1) | (cvt_e4m3x2(x2, x3) << 16);
  }
  uint8_t *dst = (is_v ? q.v_cache : q.k_cache) + (int64_t)page * q.kv_sp + (int64_t)h * q.kv_sh + (int64_t)t * q.kv_st + c;
  *reinterpret_cast<uint4 *>(dst) = make_uint4(out[0], out[1], out[2], out[3]);
}

int launch_quantize_pages(const QuantParams &qp, int n_list, cudaStream_t st, int64_t *n_launches) {
  if (n_list <= 0) return 0;
  const int64_t per_page = (int64_t)qp.H * qp.T_f * qp.d;
  dim3 grid((unsigned)((per_page / 16 + 255) / 256), n_list, 2);
  li_quantize_pages_kernel<<<grid, 256, 0, st>>>(qp);
  if (n_launches) *n_launches += 1;
  return (int)cudaGetLastError();
}

// Pooling of the historical K blocks from e4m3 pages (d == 128).  grid = (Mmax, H, B), 256 threads; a row is 128 bytes =
// 8 threads x 16 codes, 32 rows per pass, 4 passes for a 128-row block; all loads are issued before the first use.
// kbar[m] = scale[h] * (sum of the decoded codes) / |K_m|  (Eq. 9, true cardinality), stored channel-major like the bf16
// path; the codes decode exactly (e4m3 -> f16 -> f32), sums in fp32.
template <bool K3D>
__global__ void __launch_bounds__(256, 4) li_pool_k8_kernel(const SelectParams p, const BatchMeta meta) {
  constexpr int D = 128, TPR = 8, RPP = 32, kIter = 4;
  __shared__ __align__(16) float red[RPP][D];
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int m = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int r0 = threadIdx.x / TPR, cofs = (threadIdx.x % TPR) * 16;
  const int foff = meta.frame_off[b];
  const int n_hist = meta.frame_off[b + 1] - foff - p.n_cur;
  const int32_t *pages = p.frame_idx + foff;
  const Tiling tl = p.tl;
  if (m >= tl.num_blocks(n_hist, p.T_f, p.blk)) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    return;
  }
  const uint8_t *base = reinterpret_cast<const uint8_t *>(p.k_cache) + h * p.kv_sh + cofs;
  auto page_base = [&](int f) -> const uint8_t * {
    const int pg = __ldg(pages + f);
    return (unsigned)pg < (unsigned)p.n_pages ? base + (int64_t)pg * p.kv_sp : nullptr;
  };
  uint4 v[kIter];
  int nvalid;
  if constexpr (K3D) {
    const int per = tl.Hb * tl.Wb, tg = m / per, rem = m - tg * per, hb = rem / tl.Wb, wb = rem - hb * tl.Wb;
    const int nf = min(tl.bt, n_hist - tg * tl.bt), vh = min(tl.bh, tl.gh - hb * tl.bh), vw = min(tl.bw, tl.gw - wb * tl.bw);
    nvalid = nf * vh * vw;
#pragma unroll
    for (int it = 0; it < kIter; ++it) {                 // pass it = frame slice it of the block (32 rows per slice)
      const int hh = r0 >> tl.bw_log2, ww = r0 & (tl.bw - 1);
      v[it] = make_uint4(0, 0, 0, 0);
      if (it < nf && hh < vh && ww < vw) {
        const uint8_t *fb = page_base(tg * tl.bt + it);
        if (fb != nullptr) v[it] = ldg_stream16(fb + (int64_t)((hb * tl.bh + hh) * tl.gw + wb * tl.bw + ww) * p.kv_st);
      }
    }
  } else {
    const int L = n_hist * p.T_f, t0 = m * p.blk;
    nvalid = min(p.blk, L - t0);
    if (p.T_f >= p.blk) {
      // the block touches at most two pages: rows [0, split) lie in page F[pg0], the rest in page F[pg0 + 1]
      const int pg0 = t0 / p.T_f, row0 = t0 - pg0 * p.T_f, split = p.T_f - row0;
      const uint8_t *b0 = page_base(pg0), *b1 = split < nvalid ? page_base(pg0 + 1) : nullptr;
      if (b0 != nullptr) b0 += (int64_t)row0 * p.kv_st;
      if (b1 != nullptr) b1 -= (int64_t)split * p.kv_st;
#pragma unroll
      for (int it = 0; it < kIter; ++it) {
        const int r = r0 + it * RPP;
        const uint8_t *rb = r < split ? b0 : b1;
        v[it] = (r < nvalid && rb != nullptr) ? ldg_stream16(rb + (int64_t)r * p.kv_st) : make_uint4(0, 0, 0, 0);
      }
    } else {
#pragma unroll
      for (int it = 0; it < kIter; ++it) {               // frames shorter than a block: one page lookup per row
        const int r = r0 + it * RPP;
        v[it] = make_uint4(0, 0, 0, 0);
        if (r < nvalid) {
          const int t = t0 + r, pg = t / p.T_f;
          const uint8_t *rb = page_base(pg);
          if (rb != nullptr) v[it] = ldg_stream16(rb + (int64_t)(t - pg * p.T_f) * p.kv_st);
        }
      }
    }
  }
  uint64_t acc[8] = {0ull, 0ull, 0ull, 0ull, 0ull, 0ull, 0ull, 0ull};      // 16 channels as 8 packed fp32 pairs
#pragma unroll
  for (int it = 0; it < kIter; ++it) {
    const uint32_t w[4] = {v[it].x, v[it].y, v[it].z, v[it].w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float a0, a1, a2, a3;
      e4m3x2_to_f32(w[i], a0, a1);
      e4m3x2_to_f32(w[i] >> 16, a2, a3);
      acc[2 * i] = add2(acc[2 * i], pack2(a0, a1));
      acc[2 * i + 1] = add2(acc[2 * i + 1], pack2(a2, a3));
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
    *reinterpret_cast<uint4 *>(&red[r0][cofs + 4 * i]) = make_uint4((uint32_t)acc[2 * i], (uint32_t)(acc[2 * i] >> 32),
                                                                   (uint32_t)acc[2 * i + 1], (uint32_t)(acc[2 * i + 1] >> 32));
  __syncthreads();
  if (threadIdx.x < D) {
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < RPP; ++r) s += red[r][threadIdx.x];
    p.kbar[(((int64_t)b * p.H + h) * D + threadIdx.x) * p.Mp + m] = __ldg(p.k_scale + h) * (s / (float)nvalid);
  }
  // launched as a programmatic dependent of the bf16 pool kernel (query blocks), with which it shares nothing: the two
  // overlap; waiting here, after the work, makes this grid's completion imply that one's for the kernels that follow
  asm volatile("griddepcontrol.wait;" ::: "memory");
}

int launch_pool_k8(const SelectParams &sp, const BatchMeta &meta, cudaStream_t st, int64_t *n_launches) {
  if (sp.Mmax <= 0) return 0;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(sp.Mmax, sp.H, sp.B);
  cfg.blockDim = dim3(256);
  cfg.stream = st;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const cudaError_t e = sp.tl.bt > 0 ? cudaLaunchKernelEx(&cfg, li_pool_k8_kernel<true>, sp, meta)
                                      : cudaLaunchKernelEx(&cfg, li_pool_k8_kernel<false>, sp, meta);
  if (e != cudaSuccess) return (int)e;
  if (n_launches) *n_launches += 1;
  return 0;
}

}  // namespace li
