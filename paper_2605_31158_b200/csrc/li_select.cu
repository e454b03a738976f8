// li_select.cu -- li_block_select for sm_100a (Eq. 9-10).
//   kernel 1  li_pool_kernel        : block means of Q and of the historical K (K rows fetched through the
//                                     frame-index list, in place).  HBM-bound streaming reduction: every Q and
//                                     historical-K byte is read exactly once with 16-byte loads.
//   kernel 2  li_score_topk_kernel  : one CTA per 16 query-block rows of a (call, head): kbar streamed into shared memory
//                                     by bulk async copies, scores qbar_i . kbar_m / sqrt(d) (fp32, packed FMAs), then
//                                     one warp per row: the scores stay in registers as order-preserving keys, an
//                                     MSB-first radix select finds the k-th largest, ties -> lowest block index,
//                                     indices written ascending.
//   (M > 512 historical blocks: li_score_kernel writes the keys to the workspace and li_topk_kernel selects from there.)
#include <atomic>

#include "li_internal.h"
#include "li_ptx.cuh"

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
// 8 bf16 -> four packed fp32 pairs, accumulated with add.rn.f32x2 (one FADD2 per pair; a zero vector adds nothing)
__device__ __forceinline__ void add_bf16x8(uint64_t (&acc)[4], const uint4 &v) {
  acc[0] = add2(acc[0], pack2(__uint_as_float(v.x << 16), __uint_as_float(v.x & 0xffff0000u)));
  acc[1] = add2(acc[1], pack2(__uint_as_float(v.y << 16), __uint_as_float(v.y & 0xffff0000u)));
  acc[2] = add2(acc[2], pack2(__uint_as_float(v.z << 16), __uint_as_float(v.z & 0xffff0000u)));
  acc[3] = add2(acc[3], pack2(__uint_as_float(v.w << 16), __uint_as_float(v.w & 0xffff0000u)));
}

constexpr int kPoolThreads = 256;

// grid = (Nqb + Mmax, H, B).  blockIdx.x < Nqb: query block; otherwise historical K block m = x - Nqb.
// One CTA reduces one block (<= 128 rows x d).  All of a thread's loads are issued before the first use; the per-row
// address arithmetic is kept to a compare, a select and a multiply-add: the block's position in the logical sequence
// is resolved ONCE per CTA (a 1-D block spans at most two pages when T_f >= block; a 3-D block's rows are shifts and
// masks of the row index because bh * bw == 32).
template <int D, bool K3D>
__global__ void __launch_bounds__(kPoolThreads, 4) li_pool_kernel(const SelectParams p, const BatchMeta meta) {
  constexpr int TPR = D / 8;                 // threads per row (16-byte loads)
  constexpr int RPP = kPoolThreads / TPR;    // rows per pass (16 or 32: divides a 32-row frame slice)
  constexpr int kMaxIter = 128 / RPP;        // passes for the largest block (128 rows)
  __shared__ __align__(16) float red[RPP][D];
  pdl_launch_dependents();
  const int h = blockIdx.y, b = blockIdx.z;
  const int r0 = threadIdx.x / TPR, cofs = (threadIdx.x % TPR) * 8;
  const bool is_q = (int)blockIdx.x < p.Nqb;
  const int blk_id = is_q ? (int)blockIdx.x : (int)blockIdx.x - p.Nqb;
  const int foff = meta.frame_off[b];
  const int n_hist = meta.frame_off[b + 1] - foff - p.n_cur;
  const int32_t *pages = p.frame_idx + foff;
  const Tiling tl = p.tl;
  if (!is_q && blk_id >= tl.num_blocks(n_hist, p.T_f, p.blk)) return;       // m >= M_b (whole CTA exits together)
  const uint16_t *base = is_q ? p.q + b * p.q_sb + h * p.q_sh + cofs : p.k_cache + h * p.kv_sh + cofs;
  const int64_t st = is_q ? p.q_st : p.kv_st;
  // a page id outside the pool is never dereferenced: its rows count as zeros (li_validate reports the id)
  auto page_base = [&](int f) -> const uint16_t * {
    const int pg = __ldg(pages + f);
    return (unsigned)pg < (unsigned)p.n_pages ? base + (int64_t)pg * p.kv_sp : nullptr;
  };

  uint4 v[kMaxIter];
  int nvalid;
  if constexpr (K3D) {
    // 3-D blocks: row r of block (tg, hb, wb) is frame tg*bt + r/32, grid row hb*bh + (r%32)/bw, grid
    // column wb*bw + (r%32)%bw; rows outside the grid or past the region's last frame are padding (not loaded, not
    // counted: "masked loads")
    const int n_reg = is_q ? p.Lq / p.T_f : n_hist;
    const int per = tl.Hb * tl.Wb, tg = blk_id / per, rem = blk_id - tg * per, hb = rem / tl.Wb, wb = rem - hb * tl.Wb;
    const int nf = min(tl.bt, n_reg - tg * tl.bt), vh = min(tl.bh, tl.gh - hb * tl.bh), vw = min(tl.bw, tl.gw - wb * tl.bw);
    nvalid = nf * vh * vw;
    if (!is_q && p.slice_cache != nullptr) {
      // page-resident patch sums (li_pool_pages): the block mean from <= bt cached rows, one channel per thread
      if (threadIdx.x < D) {
        float s = 0.f;
        for (int f = 0; f < nf; ++f) {
          const int pg = __ldg(pages + tg * tl.bt + f);
          if ((unsigned)pg < (unsigned)p.n_pages) s += __ldg(p.slice_cache + (((int64_t)pg * p.H + h) * per + rem) * D + threadIdx.x);
        }
        p.kbar[(((int64_t)b * p.H + h) * D + threadIdx.x) * p.Mp + blk_id] = s / (float)nvalid;
      }
      return;
    }
#pragma unroll
    for (int it = 0; it < kMaxIter; ++it) {
      const int fs = (it * RPP) >> 5;                                       // frame slice of this pass (compile time)
      const int within = r0 + ((it * RPP) & 31), hh = within >> tl.bw_log2, ww = within & (tl.bw - 1);
      v[it] = make_uint4(0, 0, 0, 0);
      if (fs < nf && hh < vh && ww < vw) {
        const int f = tg * tl.bt + fs;
        const uint16_t *fb = is_q ? base + (int64_t)f * p.T_f * st : page_base(f);
        if (fb != nullptr) v[it] = ldg_stream(fb + (int64_t)((hb * tl.bh + hh) * tl.gw + wb * tl.bw + ww) * st);
      }
    }
  } else {
    const int L = is_q ? p.Lq : n_hist * p.T_f, t0 = blk_id * p.blk;
    nvalid = min(p.blk, L - t0);
    if (is_q) {
      const uint16_t *b0 = base + (int64_t)t0 * st;
#pragma unroll
      for (int it = 0; it < kMaxIter; ++it) {
        const int r = r0 + it * RPP;
        v[it] = r < nvalid ? ldg_stream(b0 + (int64_t)r * st) : make_uint4(0, 0, 0, 0);
      }
    } else if (p.T_f >= p.blk) {
      // the block touches at most two pages: rows [0, split) lie in page F[pg0], the rest in page F[pg0 + 1]
      const int pg0 = t0 / p.T_f, row0 = t0 - pg0 * p.T_f, split = p.T_f - row0;
      const uint16_t *b0 = page_base(pg0), *b1 = split < nvalid ? page_base(pg0 + 1) : nullptr;
      if (b0 != nullptr) b0 += (int64_t)row0 * st;
      if (b1 != nullptr) b1 -= (int64_t)split * st;
#pragma unroll
      for (int it = 0; it < kMaxIter; ++it) {
        const int r = r0 + it * RPP;
        const uint16_t *rb = r < split ? b0 : b1;
        v[it] = (r < nvalid && rb != nullptr) ? ldg_stream(rb + (int64_t)r * st) : make_uint4(0, 0, 0, 0);
      }
    } else {
      // frames shorter than a block: one page lookup per row
#pragma unroll
      for (int it = 0; it < kMaxIter; ++it) {
        const int r = r0 + it * RPP;
        v[it] = make_uint4(0, 0, 0, 0);
        if (r < nvalid) {
          const int t = t0 + r, pg = t / p.T_f;
          const uint16_t *rb = page_base(pg);
          if (rb != nullptr) v[it] = ldg_stream(rb + (int64_t)(t - pg * p.T_f) * st);
        }
      }
    }
  }
  uint64_t acc[4] = {0ull, 0ull, 0ull, 0ull};                              // four (+0.0f, +0.0f) pairs
#pragma unroll
  for (int it = 0; it < kMaxIter; ++it) add_bf16x8(acc, v[it]);

  *reinterpret_cast<uint4 *>(&red[r0][cofs]) = make_uint4((uint32_t)acc[0], (uint32_t)(acc[0] >> 32), (uint32_t)acc[1], (uint32_t)(acc[1] >> 32));
  *reinterpret_cast<uint4 *>(&red[r0][cofs + 4]) = make_uint4((uint32_t)acc[2], (uint32_t)(acc[2] >> 32), (uint32_t)acc[3], (uint32_t)(acc[3] >> 32));
  __syncthreads();
  if (threadIdx.x < D) {
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < RPP; ++r) s += red[r][threadIdx.x];
    const float mean = s / (float)nvalid;                                    // Eq. 9: true cardinality |Q_i|, |K_m|
    if (is_q) p.qbar[(((int64_t)b * p.H + h) * p.Nqb + blk_id) * D + threadIdx.x] = mean;
    else p.kbar[(((int64_t)b * p.H + h) * D + threadIdx.x) * p.Mp + blk_id] = mean;   // kbar is stored TRANSPOSED: [B,H,d,Mp]
  }
}

__device__ __forceinline__ uint32_t order_key(float s) {
  const uint32_t u = __float_as_uint(s);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);   // unsigned order == float order
}

// ----------------------------------------------------------------------------- fused scores + Top_k (Eq. 10), M <= 512
// One CTA = up to 16 consecutive query-block rows of one (call, head); grid = (ceil(Nqb / rows), B*H), 16 warps; rows per
// CTA are chosen on the host so that the grid fills, but stays inside, one wave of one CTA per SM where it can.
// The head's pooled keys kbar[bh] (channel-major [D][Mp], contiguous) are streamed into shared memory by bulk async
// copies (cp.async.bulk + mbarrier), one per channel quarter, all issued up front (fewer when four do not fit; the
// others follow into the slots read first): no load latency is paid per FMA and no register holds data in flight.
// Phase 1 (scores): warp w = (32-block group g = w mod nxp, channel part cp = w / nxp) holds all rows of the CTA, by
//   quads, against the 32 blocks m = 32 g + lane (nxp = Mp / 32 groups): per channel one conflict-free LDS of kbar, one
//   broadcast LDS.128 of pooled query values and 2 packed FMAs (fma.rn.f32x2: two rows per instruction) per row quad in
//   use (the loop is instantiated for 1..4 quads; addresses advance by constant steps).  The 16 / nxp channel parts take
//   interleaved channels; their partial sums go to shared memory [part][row][Mp].
// Phase 2 (Top_k): warp w owns row w: a score is the sum of its parts in a fixed order; the scores stay in registers as
//   order-preserving keys, the k-th largest is found by an MSB-first radix select (one counting pass with redux.sync per
//   bit, ending early once exactly k keys pass), and one ordered pass emits, ascending, every block above the threshold
//   plus the lowest-index blocks equal to it.
constexpr int kSelWarps = 16;
constexpr int kSelRowsMax = 16;
constexpr int kSelPartFloats = kSelRowsMax * 16 * 32;      // [parts][16 rows][Mp] with parts * Mp <= 16 * 32
__host__ __device__ inline size_t sel_smem_bytes(int D, int Mp, int n_slots) {
  return 128 + (size_t)(D * kSelRowsMax + kSelPartFloats + n_slots * (D / 4) * Mp) * sizeof(float);
}
// pooled query value (channel c, row r) lives at float c*16 + r: a warp reads 4 consecutive rows with one broadcast
// LDS.128; staged by one STS.128 per (channel, row quad)
// One channel quarter of phase 1 for a warp: channels c = cp, cp + parts, ... of the quarter, RQ row quads (4 RQ rows)
// against the 32 blocks of the warp's group; unrolled by 4 channels with the kbar loads up front.
template <int RQ>
__device__ __forceinline__ void score_quarter(const float *kq, const float *qq, int cp, int parts, int DW, int Mp,
                                              uint64_t (&acc)[kSelRowsMax / 2]) {
  const int kstep = parts * Mp, qstep = parts * kSelRowsMax;
  kq += (size_t)cp * Mp;
  qq += cp * kSelRowsMax;
  int c = cp;
  for (; c + 3 * parts < DW; c += 4 * parts) {
    float kv[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) kv[u] = kq[u * kstep];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint64_t kk = pack2(kv[u], kv[u]);
#pragma unroll
      for (int rq = 0; rq < RQ; ++rq) {
        const float4 q4 = *reinterpret_cast<const float4 *>(qq + u * qstep + 4 * rq);
        acc[2 * rq] = fma2(pack2(q4.x, q4.y), kk, acc[2 * rq]);
        acc[2 * rq + 1] = fma2(pack2(q4.z, q4.w), kk, acc[2 * rq + 1]);
      }
    }
    kq += 4 * kstep;
    qq += 4 * qstep;
  }
  for (; c < DW; c += parts) {
    const float kv = *kq;
    const uint64_t kk = pack2(kv, kv);
#pragma unroll
    for (int rq = 0; rq < RQ; ++rq) {
      const float4 q4 = *reinterpret_cast<const float4 *>(qq + 4 * rq);
      acc[2 * rq] = fma2(pack2(q4.x, q4.y), kk, acc[2 * rq]);
      acc[2 * rq + 1] = fma2(pack2(q4.z, q4.w), kk, acc[2 * rq + 1]);
    }
    kq += kstep;
    qq += qstep;
  }
}

// MINB = 1: register budget of one CTA per SM (all loads of four channels in flight), for grids inside one wave;
// MINB = 2: 64 registers, two CTAs per SM where the shared memory allows it (many calls x heads).
template <int D, int NX, int MINB>
__global__ void __launch_bounds__(kSelWarps * 32, MINB) li_score_topk_kernel(const SelectParams p, const BatchMeta meta,
                                                                        const int rows_per_cta, const int n_slots) {
  extern __shared__ __align__(128) uint8_t sel_smem[];
  constexpr int DW = D / 4;
  float *sqT = reinterpret_cast<float *>(sel_smem + 128);  // [D][16 rows]
  float *part = sqT + D * kSelRowsMax;                     // [parts][16][Mp]: partial dot products
  float *ring = part + kSelPartFloats;                     // [n_slots][DW][Mp]: channel quarters of kbar[bh]
  const uint32_t bar0 = smem_u32(sel_smem);                // 4 mbarriers, one per channel quarter (each used once)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int bh = blockIdx.y, b = bh / p.H;
  const int i0 = blockIdx.x * rows_per_cta, R = min(rows_per_cta, p.Nqb - i0);
  const int n_hist = meta.frame_off[b + 1] - meta.frame_off[b] - p.n_cur;
  const int M = p.tl.num_blocks(n_hist, p.T_f, p.blk);
  const int k = min(meta.top_k[b], M);
  const int nx = (M + 31) >> 5;                            // 32-block groups that exist (CTA-uniform), <= 16
  const int nxp = p.Mp >> 5;                               // groups the row pitch holds (>= nx, batch-uniform), <= 16
  const int parts = kSelWarps / nxp;                       // channel parts (warps per group); parts * Mp <= 16 * 32
  const bool scoring = M > 0 && (k > 0 || p.scores != nullptr);   // CTA-uniform
  const uint32_t quarter_bytes = (uint32_t)(DW * p.Mp * sizeof(float));
  const float *ksrc = p.kbar + (int64_t)bh * D * p.Mp;
  auto copy_quarter = [&](int q) {                         // one elected thread
    const uint32_t mb = bar0 + 8u * q, dst = smem_u32(ring) + (uint32_t)(q % n_slots) * quarter_bytes;
    mbar_arrive_expect_tx(mb, quarter_bytes);
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(ksrc + (size_t)q * DW * p.Mp), "r"(quarter_bytes), "r"(mb) : "memory");
  };
  if (threadIdx.x == 0) {
    for (int q = 0; q < 4; ++q) mbar_init(bar0 + 8u * q, 1);
    mbar_fence_init();
    fence_proxy_async();
  }
  pdl_launch_dependents();
  pdl_wait();                                              // qbar / kbar come from li_pool_kernel
  if (scoring) {
    if (threadIdx.x == 0)
      for (int q = 0; q < n_slots; ++q) copy_quarter(q);
    for (int t = threadIdx.x; t < (kSelRowsMax / 4) * D; t += kSelWarps * 32) {
      const int rq = t / D, c = t - rq * D;                // consecutive lanes: consecutive channels (coalesced loads)
      const float *src = p.qbar + ((int64_t)bh * p.Nqb + i0 + 4 * rq) * D + c;
      float4 v;
      v.x = 4 * rq + 0 < R ? __ldg(src) : 0.f;
      v.y = 4 * rq + 1 < R ? __ldg(src + D) : 0.f;
      v.z = 4 * rq + 2 < R ? __ldg(src + 2 * D) : 0.f;
      v.w = 4 * rq + 3 < R ? __ldg(src + 3 * D) : 0.f;
      *reinterpret_cast<float4 *>(sqT + c * kSelRowsMax + 4 * rq) = v;
    }
    __syncthreads();                                       // barriers initialised, query values staged
    const int g = warp % nxp, cp = warp / nxp;             // idle: cp >= parts (16 is not a multiple of nxp), g >= nx (short call)
    const int nrq = (rows_per_cta + 3) >> 2;               // row quads held by a CTA of this launch (1..4)
    uint64_t acc[kSelRowsMax / 2];                         // acc[rp] = (row 2 rp, row 2 rp + 1) against block 32 g + lane
#pragma unroll
    for (int rp = 0; rp < kSelRowsMax / 2; ++rp) acc[rp] = 0ull;
    for (int q = 0; q < 4; ++q) {
      mbar_wait(bar0 + 8u * q, 0);
      if (cp < parts && g < nx) {
        const float *kq = ring + (size_t)(q % n_slots) * DW * p.Mp + 32 * g + lane;
        const float *qq = sqT + (size_t)q * DW * kSelRowsMax;
        switch (nrq) {                                     // CTA-uniform: only the row quads this CTA holds
          case 1: score_quarter<1>(kq, qq, cp, parts, DW, p.Mp, acc); break;
          case 2: score_quarter<2>(kq, qq, cp, parts, DW, p.Mp, acc); break;
          case 3: score_quarter<3>(kq, qq, cp, parts, DW, p.Mp, acc); break;
          default: score_quarter<4>(kq, qq, cp, parts, DW, p.Mp, acc); break;
        }
      }
      if (q + n_slots < 4) {                               // the ring is shorter than the head: refill the slot just read
        __syncthreads();
        if (threadIdx.x == 0) copy_quarter(q + n_slots);
      }
    }
    if (cp < parts && g < nx) {
      float *pw = part + (size_t)cp * kSelRowsMax * p.Mp + 32 * g + lane;
#pragma unroll
      for (int rp = 0; rp < kSelRowsMax / 2; ++rp) {
        if (2 * rp < R) {                                  // CTA-uniform
          float s0, s1;
          unpack2(acc[rp], s0, s1);
          pw[(size_t)(2 * rp) * p.Mp] = s0;
          pw[(size_t)(2 * rp + 1) * p.Mp] = s1;
        }
      }
    }
  }
  __syncthreads();

  if (warp >= R) return;                                   // whole warp; no CTA-wide barrier below
  const int64_t row = (int64_t)bh * p.Nqb + i0 + warp;
  int32_t *out = p.sel_idx + row * p.kmax;
  if (lane == 0) p.sel_cnt[row] = k;
  uint32_t kr[NX];
  {
    // a score = its channel parts added in a fixed order (part 0 first)
    float dot[NX];
    const float *pr = part + (size_t)warp * p.Mp + lane;
#pragma unroll
    for (int x = 0; x < NX; ++x) dot[x] = (lane + 32 * x < M && scoring) ? pr[32 * x] : 0.f;
    for (int pp = 1; pp < parts; ++pp) {
      pr += (size_t)kSelRowsMax * p.Mp;
#pragma unroll
      for (int x = 0; x < NX; ++x)
        if (lane + 32 * x < M && scoring) dot[x] += pr[32 * x];
    }
#pragma unroll
    for (int x = 0; x < NX; ++x) {
      const int m = lane + 32 * x;
      kr[x] = 0u;                                          // absent blocks: key 0, below every real key
      if (m < M && scoring) {
        const float sv = dot[x] * p.inv_sqrt_d + 0.0f;     // -0 -> +0 so that equal scores have equal keys
        kr[x] = order_key(sv);
        if (p.scores != nullptr) p.scores[row * p.score_pitch + m] = sv;
      }
    }
  }
  if (k > 0) {
    // T = k-th largest key: built MSB first, keeping count(key >= T) >= k
    // (the search ends as soon as exactly k keys are >= T: that set is the answer, whatever the lower bits of the k-th)
    uint32_t T = 0;
    for (int bit = 31; bit >= 0; --bit) {
      const uint32_t cand = T | (1u << bit);
      int c0 = 0, c1 = 0;
#pragma unroll
      for (int x = 0; x < NX; x += 2) {
        c0 += kr[x] >= cand;
        if (x + 1 < NX) c1 += kr[x + 1] >= cand;
      }
      const int c = __reduce_add_sync(0xffffffffu, c0 + c1);
      if (c >= k) {
        T = cand;
        if (c == k) break;                                 // warp-uniform
      }
    }
    int c_gt = 0;
#pragma unroll
    for (int x = 0; x < NX; ++x) c_gt += kr[x] > T;
    c_gt = __reduce_add_sync(0xffffffffu, c_gt);
    int need_eq = k - c_gt;                                // ties at the threshold: lowest index first
    int pos = 0;
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int x = 0; x < NX; ++x) {
      const bool gt = kr[x] > T;
      const bool eq = kr[x] == T && T != 0u;
      const uint32_t eq_mask = __ballot_sync(0xffffffffu, eq);
      const bool take = gt || (eq && __popc(eq_mask & lt) < need_eq);
      const uint32_t take_mask = __ballot_sync(0xffffffffu, take);
      if (take) out[pos + __popc(take_mask & lt)] = lane + 32 * x;
      pos += __popc(take_mask);
      need_eq -= min(need_eq, __popc(eq_mask));
    }
  }
  for (int t = k + lane; t < p.kmax; t += 32) out[t] = -1;
}

// ----------------------------------------------------------------------------- M > 512: scores and Top_k as two launches
constexpr int kRowsPerWarp = 8;              // query-block rows scored together by one warp
constexpr int kTopkWarps = 8;                // rows (warps) per CTA of the top-k kernel
constexpr int kScoreWarps = 4;
// grid = (ceil(Mmax/32), ceil(Nqb/8), B*H), 4 warps per CTA: lane = one historical block m, warp w walks channels
// [w*D/4, (w+1)*D/4) against 8 pooled query rows broadcast from shared memory; the 4 partial sums of a score are added
// in a fixed order through shared memory.  Output: order-preserving keys [B,H,Nqb,Mmax] (+ scores).
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

// One warp per row; grid = ceil(B*H*Nqb / 8) CTAs of 8 warps; keys re-read from the workspace in every counting pass.
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
    uint32_t T = 0;
    int c_gt = 0;
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
  __shared__ __align__(16) float red[RPP][D];
  const Tiling tl = p.tl;
  const int patch = blockIdx.x, h = blockIdx.y, page = pages[blockIdx.z];
  if ((unsigned)page >= (unsigned)p.n_pages) return;                        // never read or written (li_validate reports it)
  const int hb = patch / tl.Wb, wb = patch - hb * tl.Wb;
  const int r0 = threadIdx.x / TPR, cofs = (threadIdx.x % TPR) * 8;
  uint64_t acc[4] = {0ull, 0ull, 0ull, 0ull};
  const uint16_t *base = p.k_cache + (int64_t)page * p.kv_sp + h * p.kv_sh + cofs;
#pragma unroll
  for (int it = 0; it < 32 / RPP; ++it) {
    const int r = r0 + it * RPP, hh = r >> tl.bw_log2, ww = r & (tl.bw - 1), y = hb * tl.bh + hh, x = wb * tl.bw + ww;
    if (y < tl.gh && x < tl.gw) add_bf16x8(acc, ldg_stream(base + (int64_t)(y * tl.gw + x) * p.kv_st));
  }
  *reinterpret_cast<uint4 *>(&red[r0][cofs]) = make_uint4((uint32_t)acc[0], (uint32_t)(acc[0] >> 32), (uint32_t)acc[1], (uint32_t)(acc[1] >> 32));
  *reinterpret_cast<uint4 *>(&red[r0][cofs + 4]) = make_uint4((uint32_t)acc[2], (uint32_t)(acc[2] >> 32), (uint32_t)acc[3], (uint32_t)(acc[3] >> 32));
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

constexpr size_t kSelSmemMax = 227 * 1024;
template <int D, int NX, int MINB>
static cudaError_t launch_score_topk_inst(cudaLaunchConfig_t &cfg, const SelectParams &sp, const BatchMeta &meta, int rows,
                                          int n_slots) {
  if (cfg.dynamicSmemBytes > 48 * 1024) {                  // above 48 KB the limit is raised once per device
    static std::atomic<uint64_t> attr_done{0};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const uint64_t dev_bit = 1ull << (dev & 63);
    if (!(attr_done.load(std::memory_order_acquire) & dev_bit)) {
      e = cudaFuncSetAttribute(li_score_topk_kernel<D, NX, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSelSmemMax);
      if (e != cudaSuccess) return e;
      attr_done.fetch_or(dev_bit, std::memory_order_release);
    }
  }
  return cudaLaunchKernelEx(&cfg, li_score_topk_kernel<D, NX, MINB>, sp, meta, rows, n_slots);
}
template <int D, int NX>
static cudaError_t launch_score_topk_nx(cudaLaunchConfig_t &cfg, const SelectParams &sp, const BatchMeta &meta) {
  // rows per CTA: at least the fewest CTAs per head whose rows fit 16 warps; more while the grid stays inside one wave of
  // one CTA per SM (phase 1 costs a CTA per row QUAD it holds, phase 2 runs one warp per row), rows spread evenly:
  // 49 rows x 24 heads on 148 SMs -> 6 CTAs per head of 9, 9, 9, 9, 9, 4 rows (3 quads) instead of 4 of 13 (4 quads)
  int groups = (sp.Nqb + kSelRowsMax - 1) / kSelRowsMax;
  const int n_sm = device_sm_count(), per_wave = n_sm / (sp.B * sp.H);
  if (per_wave > groups) groups = per_wave < sp.Nqb ? per_wave : sp.Nqb;
  const int rows = (sp.Nqb + groups - 1) / groups;
  groups = (sp.Nqb + rows - 1) / rows;
  int n_slots = 4;                                         // channel quarters of kbar[bh] resident at once (2 always fit)
  while (n_slots > 1 && sel_smem_bytes(D, sp.Mp, n_slots) > kSelSmemMax) --n_slots;
  cfg.gridDim = dim3(groups, sp.B * sp.H);
  cfg.blockDim = dim3(kSelWarps * 32);
  cfg.dynamicSmemBytes = sel_smem_bytes(D, sp.Mp, n_slots);
  if (groups * sp.B * sp.H <= n_sm) return launch_score_topk_inst<D, NX, 1>(cfg, sp, meta, rows, n_slots);
  return launch_score_topk_inst<D, NX, 2>(cfg, sp, meta, rows, n_slots);
}
template <int D>
static cudaError_t launch_score_topk(cudaLaunchConfig_t &cfg, const SelectParams &sp, const BatchMeta &meta) {
  if (sp.Mmax <= 128) return launch_score_topk_nx<D, 4>(cfg, sp, meta);
  if (sp.Mmax <= 192) return launch_score_topk_nx<D, 6>(cfg, sp, meta);
  if (sp.Mmax <= 256) return launch_score_topk_nx<D, 8>(cfg, sp, meta);
  if (sp.Mmax <= 416) return launch_score_topk_nx<D, 13>(cfg, sp, meta);
  return launch_score_topk_nx<D, 16>(cfg, sp, meta);
}

int launch_select(const SelectParams &sp, const BatchMeta &meta, cudaStream_t st, int64_t *n_launches) {
  {
    // FP8 pages: the bf16 pool kernel takes the query blocks only, li_pool_k8_kernel the historical K blocks
    const bool k8 = sp.k_scale != nullptr;
    dim3 grid(sp.Nqb + ((sp.skip_k || k8) ? 0 : sp.Mmax), sp.H, sp.B);
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
    if (k8 && !sp.skip_k) {
      const int e8 = launch_pool_k8(sp, meta, st, n_launches);
      if (e8 != 0) return e8;
    }
  }
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.stream = st;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (sp.Mmax <= 512) {
    cudaError_t e = sp.d == 128 ? launch_score_topk<128>(cfg, sp, meta) : launch_score_topk<64>(cfg, sp, meta);
    if (e != cudaSuccess) return (int)e;
    if (n_launches) *n_launches += 1;
    return 0;
  }
  {
    cfg.gridDim = dim3((sp.Mmax + 31) / 32, (sp.Nqb + kRowsPerWarp - 1) / kRowsPerWarp, sp.B * sp.H);
    cfg.blockDim = dim3(kScoreWarps * 32);
    cudaError_t e = sp.d == 128 ? cudaLaunchKernelEx(&cfg, li_score_kernel<128>, sp, meta)
                                : cudaLaunchKernelEx(&cfg, li_score_kernel<64>, sp, meta);
    if (e != cudaSuccess) return (int)e;
    if (n_launches) *n_launches += 1;
  }
  {
    const int64_t rows = (int64_t)sp.B * sp.H * sp.Nqb;
    cfg.gridDim = dim3((unsigned)((rows + kTopkWarps - 1) / kTopkWarps));
    cfg.blockDim = dim3(kTopkWarps * 32);
    cudaError_t e = cudaLaunchKernelEx(&cfg, li_topk_kernel, sp, meta);
    if (e != cudaSuccess) return (int)e;
    if (n_launches) *n_launches += 1;
  }
  return 0;
}

// ----------------------------------------------------------------------------- li_validate (debug, include/li.h)
// CTAs [0, n_list_ctas): 256 frame-list entries each.  Then one CTA per (call, head, query block) row of sel_idx:
// count and range checks, duplicates through a bitmap of M bits in shared memory.
__device__ __forceinline__ void report(int32_t *err, int bit, int b, int pos, int val) {
  atomicOr(&err[0], bit);
  if (atomicCAS(&err[1], 0, b + 1) == 0) { err[2] = pos; err[3] = val; }
}
constexpr int kBitmapWords = 8192;          // duplicates are checked for M <= 262144
__global__ void __launch_bounds__(256) li_validate_kernel(const ValidateParams v, const BatchMeta meta, int n_list_ctas) {
  __shared__ uint32_t bm[kBitmapWords];
  if ((int)blockIdx.x < n_list_ctas) {
    const int e = blockIdx.x * 256 + threadIdx.x;
    if (e < meta.frame_off[v.B]) {
      const int pg = v.frame_idx[e];
      if ((unsigned)pg >= (unsigned)v.n_pages) {
        int b = 0;
        while (b + 1 < v.B && meta.frame_off[b + 1] <= e) ++b;
        report(v.err, LI_BAD_PAGE_ID, b, e, pg);
      }
    }
    return;
  }
  const int64_t row = (int64_t)blockIdx.x - n_list_ctas;
  const int b = (int)(row / ((int64_t)v.H * v.Nqb));
  const int n_hist = meta.frame_off[b + 1] - meta.frame_off[b] - v.n_cur;
  const int M = v.tl.num_blocks(n_hist, v.T_f, v.blk);
  const int cnt = v.sel_cnt[row];
  const int pos0 = (int)((row - (int64_t)b * v.H * v.Nqb) * v.kmax);
  if (cnt < 0 || cnt > v.kmax || cnt > M) {
    if (threadIdx.x == 0) report(v.err, LI_BAD_SEL_CNT, b, (int)(row - (int64_t)b * v.H * v.Nqb), cnt);
    return;
  }
  const bool dup_check = M <= kBitmapWords * 32;
  if (dup_check)
    for (int w = threadIdx.x; w < (M + 31) / 32; w += 256) bm[w] = 0u;
  __syncthreads();
  const int32_t *sel = v.sel_idx + row * v.kmax;
  for (int t = threadIdx.x; t < cnt; t += 256) {
    const int m = sel[t];
    if (m < 0 || m >= M) report(v.err, LI_BAD_SEL_RANGE, b, pos0 + t, m);
    else if (dup_check && (atomicOr(&bm[m >> 5], 1u << (m & 31)) >> (m & 31)) & 1u) report(v.err, LI_BAD_SEL_DUPLICATE, b, pos0 + t, m);
  }
}

int launch_validate(const ValidateParams &vp, const BatchMeta &meta, cudaStream_t st, int64_t *n_launches) {
  cudaError_t e = cudaMemsetAsync(vp.err, 0, 4 * sizeof(int32_t), st);
  if (e != cudaSuccess) return (int)e;
  const int n_list_ctas = (meta.frame_off[vp.B] + 255) / 256;
  const int64_t rows = vp.sel_idx != nullptr ? (int64_t)vp.B * vp.H * vp.Nqb : 0;
  if (n_list_ctas + rows == 0) return 0;
  li_validate_kernel<<<(unsigned)(n_list_ctas + rows), 256, 0, st>>>(vp, meta, n_list_ctas);
  if (n_launches) *n_launches += 1;
  return (int)cudaGetLastError();
}

}  // namespace li
