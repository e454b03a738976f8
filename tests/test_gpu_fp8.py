"""GPU parity of the FP8 (E4M3) K/V-page path (include/li.h LI_FLAG_KV_FP8) against
oracle/li_fp8_oracle.py through the C-ABI binding: quantise-on-write bit-exact, block mask bit-exact up to reported
ties, attention output within the tolerance DESIGN.md c20 derives for probabilities rounded to e4m3."""
from fractions import Fraction

import numpy as np
import pytest
import torch

import li_workloads as W

pytestmark = pytest.mark.gpu

# DESIGN.md c20: the oracle mirrors the e4m3 images of Q, K and V exactly; the kernel additionally rounds every
# probability to e4m3 (relative error <= 2^-4, unbiased) before the second MMA.  On the synthetic workloads (thousands of
# comparable keys per row) that adds O(1e-3); the bar is 3x the bf16 bar of BASELINE.json.
FP8_MAX_ABS, FP8_MEAN_ABS = 6e-2, 6e-3


@pytest.fixture(scope="module")
def env():
    import paper_2605_31158_b200 as li
    from oracle import li_fp8_oracle as F
    from oracle import li_oracle as O
    from tests import parity_util as P
    return li, F, O, P


def build_fp8(li, prob, grid=None, block3d=None, flags=0):
    """Per-head scales = max |value| over the pool / 448 (fp32), pages quantised on the GPU by li_quantize_pages."""
    s = prob.spec
    dev = "cuda:0"
    ks = (prob.k_cache.float().abs().amax(dim=(0, 2, 3)) / 448.0).to(torch.float32)
    vs = (prob.v_cache.float().abs().amax(dim=(0, 2, 3)) / 448.0).to(torch.float32)
    k8 = torch.full(prob.k_cache.shape, 0x7F, dtype=torch.uint8, device=dev)        # NaN codes until written
    v8 = torch.full(prob.v_cache.shape, 0x7F, dtype=torch.uint8, device=dev)
    ctx = li.Context(prob.q.to(dev), k8, v8, torch.from_numpy(prob.frame_idx).to(dev), prob.frame_off, s.n_cur_frames,
                     s.block, grid=grid, block3d=block3d, flags=flags, k_scale=ks.to(dev), v_scale=vs.to(dev))
    pages = torch.arange(s.n_pages, dtype=torch.int32, device=dev)
    li.li_quantize_pages(ctx, prob.k_cache.to(dev), prob.v_cache.to(dev), pages)
    torch.cuda.synchronize()
    return ctx, ks.numpy(), vs.numpy()


def run_case(env, spec, flags=0, prob=None, tol=None, tiles=None):
    li, F, O, P = env
    prob = prob if prob is not None else W.build(spec)
    s = prob.spec
    ctx, ks, vs = build_fp8(li, prob, grid=s.grid, block3d=s.block3d, flags=flags)
    # quantise-on-write: bit-exact codes
    kf, vf = O.widen(prob.u16(prob.k_cache)), O.widen(prob.u16(prob.v_cache))
    kc, vc = F.quantize(kf, ks, 1), F.quantize(vf, vs, 1)
    assert np.array_equal(ctx.k_cache.cpu().numpy(), kc) and np.array_equal(ctx.v_cache.cpu().numpy(), vc)
    buf = li.Buffers(ctx, prob.kmax, want_scores=True)
    buf.o.fill_(float("nan"))
    li.forward(ctx, prob.top_k, buf)
    torch.cuda.synchronize()
    if s.block3d is not None:
        osel, osc = O.block_select_3d(prob.u16(prob.q), F.dequantize(kc, ks, 1), prob.frame_idx, prob.frame_off, s.n_cur_frames,
                                      *s.grid, *s.block3d, prob.top_k)
    else:
        osel, osc = F.block_select_fp8(prob.u16(prob.q), kc, ks, prob.frame_idx, prob.frame_off, s.n_cur_frames, s.block,
                                       s.block, prob.top_k)
    excused = P.check_selection(prob, buf, osel, osc)
    gsel = [g[0] for g in P.gpu_selection(prob, buf)]
    if s.block3d is not None:
        o_ref, lse_ref = O.sparse_attn_3d(F.quantize_query_rows(prob.u16(prob.q)), F.dequantize(kc, ks, 1), F.dequantize(vc, vs, 1),
                                          prob.frame_idx, prob.frame_off, s.n_cur_frames, *s.grid, *s.block3d, gsel)
    else:
        o_ref, lse_ref = F.sparse_attn_fp8(prob.u16(prob.q), kc, vc, ks, vs, prob.frame_idx, prob.frame_off, s.n_cur_frames,
                                           s.block, s.block, gsel, tiles=tiles)
    og = buf.o.float().cpu().numpy()
    assert np.isfinite(og).all()
    lg = buf.lse.cpu().numpy()
    if tiles is not None:
        keep = ~np.isnan(lse_ref)
        og, o_ref, lg, lse_ref = og[keep], o_ref[keep], lg[keep], lse_ref[keep]
    diff = np.abs(og - o_ref)
    # always: an output is a convex combination of V rows whose weights are each off by at most 2^-4 relative
    assert diff.max() <= 2.0 ** -4 * np.abs(F.dequantize(vc, vs, 1)).max() + 1e-2
    max_abs, mean_abs = tol if tol is not None else (FP8_MAX_ABS, FP8_MEAN_ABS)
    assert diff.max() <= max_abs and diff.mean() <= mean_abs, (diff.max(), diff.mean())
    assert np.abs(lg - lse_ref).max() <= P.LSE_ABS                               # LSE sees no probability rounding
    print(f"{s.name}: excused={excused} max-abs={diff.max():.3g} mean-abs={diff.mean():.3g}")
    return prob, ctx, buf


@pytest.mark.parametrize("T_f", [200, 1560, 64])
def test_fp8_pages_full_parity_1d(env, T_f):
    """1-D blocks straddling frames (8-row TMA pieces of 128-byte e4m3 rows), ragged tails, unsorted memory pages."""
    n_cur = 1 if T_f == 1560 else 3
    spec = W.spec_small(name=f"fp8-t{T_f}", H=2, d=128, block=128, frame_tokens=T_f, n_cur_frames=n_cur, n_pages=12,
                        n_mem=(2,), n_win=(3,) if T_f != 1560 else (1,), density=Fraction(1, 2))
    run_case(env, spec)


def test_fp8_pages_3d_blocks_and_split(env):
    """3-D (4,8,4) blocks with bottom-border tiles and the tail-wave split: 5-D TMA boxes of e4m3 bytes."""
    li = env[0]
    spec = W.spec_small(name="fp8-3d", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=3, n_pages=24, n_mem=(6,),
                        n_win=(14,), density=Fraction(1, 1), grid=(10, 20), block3d=(4, 8, 4))
    li.lib().li_reset_launch_count()
    prob, ctx, buf = run_case(env, spec)
    assert li.lib().li_launch_count() == 1 + 5      # quantise | Q pool, K pool (fp8), score + top-k, attention (split), merge


def test_fp8_pages_right_border_blocks(env):
    """(4,4,8) blocks on a grid whose width is not a multiple of 8: column-masked border tiles with e4m3 pages."""
    spec = W.spec_small(name="fp8-3d-448", H=2, d=128, block=128, frame_tokens=10 * 12, n_cur_frames=4, n_pages=14, n_mem=(2,),
                        n_win=(3,), density=Fraction(1, 2), grid=(10, 12), block3d=(4, 4, 8))
    run_case(env, spec)


def test_fp8_varlen_batch_and_growing_maximum(env):
    """Several calls of different length in one launch; later pages up to 4.6x louder, so the lazy rescale path runs with
    e4m3 P.  The louder keys make the softmax rows peaky (a handful of keys carry a row), where the rounding of P no
    longer averages out: only the rigorous bound 2^-4 max|v| and a loose mean bar apply (DESIGN.md c20)."""
    spec = W.spec_small(name="fp8-batch", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=40,
                        n_mem=(0, 2, 0, 3), n_win=(1, 2, 4, 1), density=Fraction(1, 1), pages_per_call=10)
    li, F, O, P = env
    prob = W.build(spec)
    for pg in range(spec.n_pages):
        prob.k_cache[pg] = (prob.k_cache[pg].float() * (1.0 + 0.4 * (pg % 10))).to(torch.bfloat16)
    run_case(env, spec, prob=prob, tol=(0.3, 2e-2))


def test_fp8_rejections(env):
    li = env[0]
    spec = W.spec_small(name="fp8-rej", H=2, d=64, block=64, frame_tokens=64, n_cur_frames=1, n_pages=6, n_mem=(1,), n_win=(1,))
    prob = W.build(spec)
    k8 = torch.zeros(prob.k_cache.shape, dtype=torch.uint8, device="cuda")
    sc = torch.ones(2, dtype=torch.float32, device="cuda")
    ctx = li.Context(prob.q.cuda(), k8, k8.clone(), torch.from_numpy(prob.frame_idx).cuda(), prob.frame_off, 1, 64,
                     k_scale=sc, v_scale=sc)
    with pytest.raises(li.LiError) as e:
        ctx.workspace_bytes(4)                       # d = 64 is not supported with FP8 pages (li_workspace_bytes -> 0)
    with pytest.raises(ValueError):
        li.Context(prob.q.cuda(), k8, k8.clone(), torch.from_numpy(prob.frame_idx).cuda(), prob.frame_off, 1, 64)   # no scales


@pytest.mark.slow
def test_fp8_mid_shapes_two_waves_stratified(env):
    """`mid` shapes (12 heads: 588 attention CTAs = 2 waves of 2 CTAs per SM) with FP8 pages: whole mask against the
    oracle, attention on every 8th (head, query block) tile plus every ragged last block."""
    prob = W.build(W.spec_mid(H=12))
    tiles = sorted({(0, h, i) for h in range(12) for i in range(prob.Nqb) if (h + i) % 8 == 0} | {(0, h, prob.Nqb - 1) for h in range(12)})
    run_case(env, prob.spec, prob=prob, tiles=tiles)
