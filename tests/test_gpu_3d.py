"""GPU parity for the paper's 3-D block tiling (B_t,B_h,B_w) against oracle/li_oracle.py *_3d."""
from fractions import Fraction

import numpy as np
import pytest
import torch

import li_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    from tests import parity_util
    return parity_util


def small3d(name, grid, block3d, n_cur, n_mem, n_win, H=2, d=128, density=Fraction(1, 2), n_pages=14, **kw):
    gh, gw = grid
    bt, bh, bw = block3d
    return W.spec_small(name=name, H=H, d=d, block=bt * bh * bw, frame_tokens=gh * gw, n_cur_frames=n_cur,
                        n_pages=n_pages, n_mem=n_mem, n_win=n_win, density=density, grid=grid, block3d=block3d, **kw)


@pytest.mark.parametrize("grid,block3d,n_cur,n_hist", [((30, 52), (4, 8, 4), 4, (2, 4)),     # paper geometry, partial rows
                                                        ((10, 16), (4, 4, 8), 4, (3, 3)),     # Matrix-Game block shape
                                                        ((12, 8), (2, 8, 4), 2, (2, 3)),      # 64-token blocks, partial group
                                                        ((6, 8), (4, 8, 4), 3, (1, 4)),       # grid lower than a block, partial groups
                                                        ((30, 52), (4, 4, 8), 4, (2, 4)),     # Matrix-Game shape on the 52-wide grid
                                                        ((9, 24), (4, 2, 16), 2, (3, 2))])    # 16-wide blocks: 8 of 16 columns at the border
def test_select_3d(P, grid, block3d, n_cur, n_hist):
    spec = small3d(f"s3d-{grid}-{block3d}", grid, block3d, n_cur, (n_hist[0],), (n_hist[1],))
    prob = W.build(spec)
    excused = P.select_parity(prob)
    print(f"{spec.name}: M={prob.M(0)} Nqb={prob.Nqb} k={int(prob.top_k[0])} excused={excused}")


@pytest.mark.parametrize("grid,block3d,n_cur,n_hist,d", [((30, 52), (4, 8, 4), 4, (2, 4), 128),   # paper geometry: rows 24..29 partial
                                                          ((10, 16), (4, 4, 8), 4, (3, 3), 128),   # (4,4,8), partial group (6 frames)
                                                          ((12, 8), (2, 8, 4), 2, (2, 3), 64),     # 64-token blocks, d=64
                                                          ((6, 8), (4, 8, 4), 3, (1, 4), 128),     # partial chunk group (3 of 4 frames)
                                                          ((30, 52), (4, 4, 8), 4, (2, 4), 128),   # (4,4,8) on 30 x 52: right AND bottom borders
                                                          ((10, 12), (2, 4, 8), 2, (2, 3), 64),    # 64-token blocks, 4-of-8-column border
                                                          ((9, 24), (4, 2, 16), 2, (3, 2), 128)])  # 16-wide blocks, 1-row bottom border
def test_full_parity_3d(P, grid, block3d, n_cur, n_hist, d):
    """li_block_select + li_sparse_attn with 3-D blocks, element by element against the oracle: 5-D TMA boxes, zero
    filled grid rows / missing frames masked out, outputs scattered back to linear token order."""
    H = 1 if grid == (30, 52) else 2
    spec = small3d(f"f3d-{grid}-{block3d}", grid, block3d, n_cur, (n_hist[0],), (n_hist[1],), H=H, d=d)
    prob = W.build(spec)
    excused, mx, mean = P.full_parity(prob)
    print(f"{spec.name}: M={prob.M(0)} Nqb={prob.Nqb} k={int(prob.top_k[0])} excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_3d_dense_and_chunk_only(P):
    """r = 1 -> dense attention over the whole context (torch SDPA); k = 0 -> chunk-only attention."""
    for density, name in ((Fraction(1, 1), "dense"), (None, "k0")):
        spec = small3d(f"f3d-{name}", (10, 16), (4, 8, 4), 4, (1,), (2,), density=density or Fraction(1, 2),
                       **({"top_k": 0} if density is None else {}))
        prob = W.build(spec)
        ctx, buf = P.run_gpu(prob)
        frames = prob.frame_idx if density is not None else prob.frame_idx[-4:]
        K = torch.cat([prob.k_cache[int(p)] for p in frames], dim=1).float()
        V = torch.cat([prob.v_cache[int(p)] for p in frames], dim=1).float()
        ref = torch.nn.functional.scaled_dot_product_attention(prob.q[0].float(), K, V)
        diff = (buf.o[0].float().cpu() - ref).abs()
        assert torch.isfinite(buf.o.float()).all() and diff.max() <= P.MAX_ABS and diff.mean() <= P.MEAN_ABS


@pytest.mark.parametrize("mode,Lt", [("1d", 77), ("1d", 40), ("1d", 256), ("3d", 77), ("3d", 136)])
def test_text_prefix_is_always_attended(P, mode, Lt):
    """T of Eq. 11: a dense text K/V region attended by every query block on top of the chunk and
    the selected history; ragged text tail, text shorter than one half-tile, strided text tensor."""
    import paper_2605_31158_b200 as li
    from oracle import li_oracle as O
    if mode == "1d":
        spec = W.spec_small(name="text-1d", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=10,
                            n_mem=(2,), n_win=(2,), density=Fraction(1, 2))
    else:
        spec = small3d("text-3d", (10, 16), (4, 8, 4), 4, (2,), (3,))
    prob = W.build(spec)
    g = torch.Generator().manual_seed(1000 + Lt)
    wide = torch.randn((1, spec.H, Lt, 2 * spec.d), generator=g).to(torch.bfloat16)       # [..., :d] = K, [..., d:] = V
    tk, tv = wide[..., :spec.d], wide[..., spec.d:]                                        # token stride 2d
    dev = "cuda:0"
    wide_d = wide.to(dev)
    ctx = li.Context(prob.q.to(dev), prob.k_cache.to(dev), prob.v_cache.to(dev), torch.from_numpy(prob.frame_idx).to(dev),
                     prob.frame_off, spec.n_cur_frames, spec.block, grid=spec.grid, block3d=spec.block3d,
                     text_k=wide_d[..., :spec.d], text_v=wide_d[..., spec.d:])
    buf = li.Buffers(ctx, prob.kmax, want_scores=True)
    buf.o.fill_(float("nan"))
    li.forward(ctx, prob.top_k, buf)
    torch.cuda.synchronize()
    osel, osc = P.oracle_select(prob)                      # text takes no part in pooling / selection
    P.check_selection(prob, buf, osel, osc)
    gsel = [g_[0] for g_ in P.gpu_selection(prob, buf)]
    u16 = lambda t: t.contiguous().view(torch.int16).numpy().view(np.uint16)
    s = spec
    if s.block3d is not None:
        o_ref, lse_ref = O.sparse_attn_3d(prob.u16(prob.q), prob.u16(prob.k_cache), prob.u16(prob.v_cache), prob.frame_idx,
                                          prob.frame_off, s.n_cur_frames, *s.grid, *s.block3d, gsel,
                                          text_k=u16(tk), text_v=u16(tv))
    else:
        o_ref, lse_ref = O.sparse_attn(prob.u16(prob.q), prob.u16(prob.k_cache), prob.u16(prob.v_cache), prob.frame_idx,
                                       prob.frame_off, s.n_cur_frames, s.block, s.block, gsel,
                                       text_k=u16(tk), text_v=u16(tv))
    mx, mean = P.compare_output(buf.o, buf.lse, o_ref, lse_ref)
    print(f"text {mode} Lt={Lt}: max-abs {mx:.3g} mean-abs {mean:.3g}")


def test_3d_more_tiles_than_the_shared_memory_tables_hold(P):
    """One query block attending 2150 selected 3-D blocks (+1 chunk block): more tiles than the per-CTA geometry table
    (2048), the selected-index table (1024) and the frame table (256) hold, so the global-memory fallbacks run; the
    single query block is also shared by 8 CTAs (tail-wave split).  Pages repeat, so ties are exact: bit-identical mask."""
    import paper_2605_31158_b200 as li
    from oracle import li_oracle as O
    g = torch.Generator().manual_seed(23)
    H, d, gh, gw, bt, bh, bw = 1, 64, 8, 4, 4, 8, 4
    T_f, n_hist, k = gh * gw, 4 * 2200, 2150
    q = torch.randn((1, H, 4 * T_f, d), generator=g).to(torch.bfloat16)
    kc = torch.randn((12, H, T_f, d), generator=g).to(torch.bfloat16)
    vc = torch.randn((12, H, T_f, d), generator=g).to(torch.bfloat16)
    fi = np.concatenate([torch.randint(0, 8, (n_hist,), generator=g).numpy(), [8, 9, 10, 11]]).astype(np.int32)
    fo = np.asarray([0, n_hist + 4], np.int32)
    ctx = li.Context(q.cuda(), kc.cuda(), vc.cuda(), torch.from_numpy(fi).cuda(), fo, 4, 128, grid=(gh, gw),
                     block3d=(bt, bh, bw))
    assert ctx.Nqb == 1 and ctx.Mmax == 2200
    buf = li.Buffers(ctx, k, want_scores=True)
    li.lib().li_reset_launch_count()
    li.forward(ctx, [k], buf)
    torch.cuda.synchronize()
    assert li.lib().li_launch_count() == 5           # M > 512: pool, scores, top-k, attention (split), merge
    u16 = lambda t: t.view(torch.int16).numpy().view(np.uint16)
    osel, osc = O.block_select_3d(u16(q), u16(kc), fi, fo, 4, gh, gw, bt, bh, bw, [k])
    np.testing.assert_array_equal(buf.sel_idx.cpu().numpy()[0], osel[0])
    o_ref, lse_ref = O.sparse_attn_3d(u16(q), u16(kc), u16(vc), fi, fo, 4, gh, gw, bt, bh, bw, osel)
    P.compare_output(buf.o, buf.lse, o_ref, lse_ref)


@pytest.mark.parametrize("grid,block3d,n_cur,n_hist,d", [((30, 52), (4, 8, 4), 4, (2, 4), 128),   # paper geometry, border patches
                                                          ((10, 16), (4, 4, 8), 4, (3, 3), 128),   # (4,4,8), partial group
                                                          ((12, 8), (2, 8, 4), 2, (2, 3), 64),     # 64-token blocks, d = 64
                                                          ((6, 8), (4, 8, 4), 3, (1, 4), 128)])    # grid lower than a patch
def test_select_from_page_resident_patch_sums(P, grid, block3d, n_cur, n_hist, d):
    """li_pool_pages + li_block_select_cached (include/li.h): historical block means formed from per-page patch sums
    must give the oracle's scores and mask, also after a page was rewritten and re-pooled alone, and for a batch of
    calls sharing the page pool."""
    import paper_2605_31158_b200 as li
    spec = small3d(f"s3d-cache-{grid}-{block3d}", grid, block3d, n_cur, (n_hist[0], 0, 1), (n_hist[1], 2, 3), d=d,
                   n_pages=42, pages_per_call=14)
    prob = W.build(spec)
    ctx = P.upload(prob)
    buf = li.Buffers(ctx, prob.kmax, want_scores=True)
    cache = torch.full((li.li_slice_cache_bytes(ctx) // 4,), float("nan"), dtype=torch.float32, device="cuda")
    li.li_pool_pages(ctx, torch.arange(spec.n_pages, dtype=torch.int32, device="cuda"), cache)
    for rewrite in (False, True):
        if rewrite:          # the model rewrites one historical page of call 0: only that page is pooled again
            pg = int(prob.frame_idx[0])
            g = torch.Generator().manual_seed(99)
            prob.k_cache[pg] = torch.randn(prob.k_cache[pg].shape, generator=g).to(torch.bfloat16)
            ctx.k_cache[pg].copy_(prob.k_cache[pg])
            li.li_pool_pages(ctx, torch.tensor([pg], dtype=torch.int32, device="cuda"), cache)
        buf.sel_idx.fill_(-7)
        li.li_block_select_cached(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, cache, buf.workspace, buf.scores)
        torch.cuda.synchronize()
        osel, osc = P.oracle_select(prob)
        excused = P.check_selection(prob, buf, osel, osc)
        # and the direct path on the same data: same scores up to the fp32 summation order
        sc_cached = buf.scores.clone()
        li.li_block_select(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, buf.workspace, buf.scores)
        torch.cuda.synchronize()
        for b in range(prob.B):
            M = prob.M(b)
            torch.testing.assert_close(sc_cached[b, :, :, :M], buf.scores[b, :, :, :M], rtol=1e-5, atol=1e-6)
    print(f"cached select {grid} {block3d}: excused={excused}")


def test_text_prefix_3d_with_tail_wave_split(P):
    """Text prefix + 3-D blocks + split query blocks in one launch (the TEXT x K3D x SPLIT kernel instance)."""
    import paper_2605_31158_b200 as li
    from oracle import li_oracle as O
    spec = small3d("text-3d-split", (10, 16), (4, 8, 4), 4, (8,), (12,), density=Fraction(1, 1), n_pages=30)
    prob = W.build(spec)
    Lt = 200
    g = torch.Generator().manual_seed(777)
    tk = torch.randn((1, spec.H, Lt, spec.d), generator=g).to(torch.bfloat16)
    tv = torch.randn((1, spec.H, Lt, spec.d), generator=g).to(torch.bfloat16)
    ctx = li.Context(prob.q.cuda(), prob.k_cache.cuda(), prob.v_cache.cuda(), torch.from_numpy(prob.frame_idx).cuda(),
                     prob.frame_off, spec.n_cur_frames, spec.block, grid=spec.grid, block3d=spec.block3d,
                     text_k=tk.cuda(), text_v=tv.cuda())
    buf = li.Buffers(ctx, prob.kmax, want_scores=True)
    buf.o.fill_(float("nan"))
    li.lib().li_reset_launch_count()
    li.forward(ctx, prob.top_k, buf)
    torch.cuda.synchronize()
    assert li.lib().li_launch_count() == 4, "split not taken"
    osel, osc = P.oracle_select(prob)
    P.check_selection(prob, buf, osel, osc)
    gsel = [g_[0] for g_ in P.gpu_selection(prob, buf)]
    u16 = lambda t: t.contiguous().view(torch.int16).numpy().view(np.uint16)
    s = spec
    o_ref, lse_ref = O.sparse_attn_3d(prob.u16(prob.q), prob.u16(prob.k_cache), prob.u16(prob.v_cache), prob.frame_idx,
                                      prob.frame_off, s.n_cur_frames, *s.grid, *s.block3d, gsel, text_k=u16(tk), text_v=u16(tv))
    mx, mean = P.compare_output(buf.o, buf.lse, o_ref, lse_ref)
    print(f"text-3d-split: max-abs {mx:.3g} mean-abs {mean:.3g}")
