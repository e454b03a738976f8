"""GPU parity tests (-m gpu): the CUDA path, called through the C-ABI binding, against oracle/li_oracle.py on the
same seeded inputs.  Bars (BASELINE.json north_star): block mask bit-exact except reported ties within 1e-4
relative of the k-th score; attention output max-abs <= 2e-2 and mean-abs <= 2e-3 against the oracle."""
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


def test_tiny_config_full_parity(P):
    """BASELINE.json configs[0]: B=1,H=2,d=64,T_f=256,Lq=256, frames {0,3}|{6}|{7}, block 64, top-k 8."""
    prob = W.build(W.spec_tiny())
    assert prob.M(0) == 12 and prob.Nqb == 4 and int(prob.top_k[0]) == 8
    excused, mx, mean = P.full_parity(prob)
    print(f"tiny: excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


@pytest.mark.parametrize("d,block,T_f", [(128, 128, 200), (64, 128, 200), (128, 64, 72), (64, 64, 40), (128, 128, 1560)])
def test_small_full_parity_straddling_blocks(P, d, block, T_f):
    """Reduced shapes: T_f not a multiple of the block (blocks straddle frames, 8-row TMA pieces), ragged
    history and chunk tails, unsorted memory pages, several query tiles."""
    n_cur = 1 if T_f == 1560 else 3
    spec = W.spec_small(name=f"small-d{d}-b{block}-t{T_f}", H=2, d=d, block=block, frame_tokens=T_f,
                        n_cur_frames=n_cur, n_pages=12, n_mem=(2,), n_win=(3,) if T_f != 1560 else (1,),
                        density=Fraction(1, 2))
    prob = W.build(spec)
    excused, mx, mean = P.full_parity(prob)
    print(f"{spec.name}: M={prob.M(0)} k={int(prob.top_k[0])} excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_small_varlen_batch_and_no_memory_calls(P):
    """adaptive-like: several independent calls in one launch, ragged Lk, calls without retrieved memory."""
    spec = W.spec_small(name="small-adaptive", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=2,
                        n_pages=40, n_mem=(0, 2, 0, 3), n_win=(1, 2, 4, 1), density=Fraction(3, 10),
                        pages_per_call=10)
    prob = W.build(spec)
    assert prob.B == 4 and len(set(prob.M(b) for b in range(4))) > 1
    excused, mx, mean = P.full_parity(prob)
    print(f"small-adaptive: excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_dense_equivalence_small(P):
    """r = 1: every block selected -> equals dense attention over the whole gathered context (torch SDPA on CPU,
    fp32, as an independent library routine) and the oracle."""
    spec = W.spec_small(name="small-dense", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=2,
                        n_pages=10, n_mem=(2,), n_win=(2,), density=Fraction(1, 1))
    prob = W.build(spec)
    ctx, buf = P.run_gpu(prob)
    M = prob.M(0)
    sel = buf.sel_idx.cpu().numpy()[0]
    assert (sel == np.arange(M)).all()
    frames = prob.frame_idx
    K = torch.cat([prob.k_cache[int(p)] for p in frames], dim=1).float()     # [H, Lk, d]
    V = torch.cat([prob.v_cache[int(p)] for p in frames], dim=1).float()
    ref = torch.nn.functional.scaled_dot_product_attention(prob.q[0].float(), K, V)
    diff = (buf.o[0].float().cpu() - ref).abs()
    assert diff.max() <= P.MAX_ABS and diff.mean() <= P.MEAN_ABS


def test_degenerate_topk_zero_and_no_history(P):
    """k = 0 -> chunk-only attention; a call with no history frames at all (M = 0)."""
    spec = W.spec_small(name="small-k0", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=10,
                        n_mem=(1, 0), n_win=(2, 0), top_k=0, pages_per_call=5)
    prob = W.build(spec)
    assert prob.M(1) == 0
    ctx, buf = P.run_gpu(prob)
    assert (buf.sel_cnt == 0).all() and (buf.sel_idx == -1).all()
    o_ref, lse_ref = P.oracle_attn(prob, [np.zeros((2, prob.Nqb, 0), np.int32)] * 2)
    P.compare_output(buf.o, buf.lse, o_ref, lse_ref)


def test_no_chunk_history_only_and_softmax_scale(P):
    """n_cur_frames = 0 (the API's 'other reading' of density): queries attend selected history only."""
    import paper_2605_31158_b200 as li
    from oracle import li_oracle as O
    g = torch.Generator().manual_seed(99)
    H, d, T_f, blk, Lq = 2, 128, 200, 128, 300
    q = torch.randn((1, H, Lq, d), generator=g).to(torch.bfloat16)
    kc = torch.randn((5, H, T_f, d), generator=g).to(torch.bfloat16)
    vc = torch.randn((5, H, T_f, d), generator=g).to(torch.bfloat16)
    fi = np.asarray([3, 1, 4], np.int32)
    fo = np.asarray([0, 3], np.int32)
    ctx = li.Context(q.cuda(), kc.cuda(), vc.cuda(), torch.from_numpy(fi).cuda(), fo, 0, blk, softmax_scale=0.05)
    buf = li.Buffers(ctx, 3, want_scores=True)
    li.forward(ctx, [3], buf)
    torch.cuda.synchronize()
    u16 = lambda t: t.view(torch.int16).numpy().view(np.uint16)
    osel, osc = O.block_select(u16(q), u16(kc), fi, fo, 0, blk, blk, [3])
    np.testing.assert_array_equal(buf.sel_idx.cpu().numpy()[0], osel[0])
    o_ref, lse_ref = O.sparse_attn(u16(q), u16(kc), u16(vc), fi, fo, 0, blk, blk, osel, softmax_scale=0.05)
    P.compare_output(buf.o, buf.lse, o_ref, lse_ref)


def test_exact_ties_lowest_index_and_page_permutation(P):
    """Duplicate page ids -> bit-identical pooled blocks -> exact ties: the GPU must pick the lowest index.
    Permuting the pool and rewriting the list must give bit-identical GPU results (gather correctness)."""
    import paper_2605_31158_b200 as li
    g = torch.Generator().manual_seed(5)
    H, d, T_f, blk = 2, 64, 64, 64
    q = torch.randn((1, H, T_f, d), generator=g).to(torch.bfloat16)
    kc = torch.randn((4, H, T_f, d), generator=g).to(torch.bfloat16)
    vc = torch.randn((4, H, T_f, d), generator=g).to(torch.bfloat16)
    fi = np.asarray([1, 0, 1, 0, 1, 2], np.int32)
    fo = np.asarray([0, 6], np.int32)

    def run(kc_, vc_, fi_, k):
        ctx = li.Context(q.cuda(), kc_.cuda(), vc_.cuda(), torch.from_numpy(fi_).cuda(), fo, 1, blk)
        buf = li.Buffers(ctx, 5, want_scores=True)
        li.forward(ctx, [k], buf)
        torch.cuda.synchronize()
        return buf

    b1 = run(kc, vc, fi, 1)
    sc = b1.scores.cpu().numpy()[0, :, 0]
    for h in range(H):
        assert sc[h, 0] == sc[h, 2] == sc[h, 4] and sc[h, 1] == sc[h, 3]
        assert int(b1.sel_idx[0, h, 0, 0]) == (0 if sc[h, 0] >= sc[h, 1] else 1)
    b2 = run(kc, vc, fi, 2)
    for h in range(H):
        assert b2.sel_idx[0, h, 0, :2].tolist() == ([0, 2] if sc[h, 0] >= sc[h, 1] else [1, 3])
    perm = torch.tensor([2, 0, 3, 1])
    inv = torch.argsort(perm).numpy()
    b3 = run(kc[perm], vc[perm], inv[fi].astype(np.int32), 2)
    assert torch.equal(b2.sel_idx, b3.sel_idx) and torch.equal(b2.o, b3.o) and torch.equal(b2.scores, b3.scores)


def test_constant_v_and_nan_in_unused_pages(P):
    """V constant -> O equals it for any mask; pages not on the frame list are NaN and must never be touched."""
    import paper_2605_31158_b200 as li
    spec = W.spec_small(name="small-nan", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=12,
                        n_mem=(2,), n_win=(2,), density=Fraction(1, 2))
    prob = W.build(spec)
    used = set(int(p) for p in prob.frame_idx)
    for pg in range(spec.n_pages):
        if pg not in used:
            prob.k_cache[pg] = float("nan")
            prob.v_cache[pg] = float("nan")
    for pg in used:
        prob.v_cache[pg] = 0.75
    ctx, buf = P.run_gpu(prob)
    o = buf.o.float().cpu()
    assert torch.isfinite(o).all() and (o - 0.75).abs().max() < 1e-2
    assert torch.isfinite(buf.scores.cpu()[..., :prob.M(0)]).all()


def test_growing_row_maximum_exercises_lazy_rescale(P):
    """Keys whose logits grow from tile to tile (later pages scaled up) force the kernel's lazy-rescale path
    (reference maximum moved, O rescaled in TMEM while earlier P.V products are still being accumulated)."""
    spec = W.spec_small(name="small-rescale", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=3, n_pages=12,
                        n_mem=(2,), n_win=(3,), density=Fraction(1, 1))
    prob = W.build(spec)
    frames = [int(x) for x in prob.frame_idx]
    # attention order is chunk blocks first, then history blocks ascending: make each later frame "louder"
    order = frames[-spec.n_cur_frames:] + frames[:-spec.n_cur_frames]
    for rank, pg in enumerate(order):
        prob.k_cache[pg] = (prob.k_cache[pg].float() * (1.0 + 1.5 * rank)).to(torch.bfloat16)
    excused, mx, mean = P.full_parity(prob)
    print(f"small-rescale: excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_strided_q_and_token_major_cache(P):
    """The ABI takes arbitrary (multiple-of-8) strides: Q as a slice of a wider tensor, the cache stored token-major
    ([page, token, head, d]) and viewed as [page, head, token, d]."""
    import paper_2605_31158_b200 as li
    spec = W.spec_small(name="small-strided", H=3, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=10,
                        n_mem=(2,), n_win=(2,), density=Fraction(1, 2))
    prob = W.build(spec)
    dev = "cuda:0"
    q_wide = torch.zeros((1, spec.H, prob.Lq, 2 * spec.d), dtype=torch.bfloat16, device=dev)
    q_wide[..., :spec.d] = prob.q.to(dev)
    q_wide[..., spec.d:] = float("nan")                                      # must never be read
    q = q_wide[..., :spec.d]
    kc = prob.k_cache.to(dev).permute(0, 2, 1, 3).contiguous().permute(0, 2, 1, 3)   # same values, token-major memory
    vc = prob.v_cache.to(dev).permute(0, 2, 1, 3).contiguous().permute(0, 2, 1, 3)
    assert q.stride(2) == 2 * spec.d and kc.stride(2) == spec.H * spec.d and kc.stride(1) == spec.d
    ctx = li.Context(q, kc, vc, torch.from_numpy(prob.frame_idx).to(dev), prob.frame_off, spec.n_cur_frames, spec.block)
    buf = li.Buffers(ctx, prob.kmax, want_scores=True)
    li.forward(ctx, prob.top_k, buf)
    torch.cuda.synchronize()
    osel, osc = P.oracle_select(prob)
    P.check_selection(prob, buf, osel, osc)
    o_ref, lse_ref = P.oracle_attn(prob, [g[0] for g in P.gpu_selection(prob, buf)])
    P.compare_output(buf.o, buf.lse, o_ref, lse_ref)


def test_many_blocks_long_lists_and_massive_ties(P):
    """M = 1200 historical blocks drawn (with repetition) from 6 pages: exact score ties everywhere (lowest index must
    win), top-k above the register fast path (M > 512), more selected blocks than the kernel stages in shared memory
    (k = 1100 > 1024) and a frame list longer than its shared-memory copy (1201 > 256)."""
    import paper_2605_31158_b200 as li
    from oracle import li_oracle as O
    g = torch.Generator().manual_seed(11)
    H, d, T_f, blk, n_hist, k = 1, 64, 64, 64, 1200, 1100
    q = torch.randn((1, H, T_f, d), generator=g).to(torch.bfloat16)
    kc = torch.randn((7, H, T_f, d), generator=g).to(torch.bfloat16)
    vc = torch.randn((7, H, T_f, d), generator=g).to(torch.bfloat16)
    fi = np.concatenate([torch.randint(0, 6, (n_hist,), generator=g).numpy(), [6]]).astype(np.int32)
    fo = np.asarray([0, n_hist + 1], np.int32)
    ctx = li.Context(q.cuda(), kc.cuda(), vc.cuda(), torch.from_numpy(fi).cuda(), fo, 1, blk)
    buf = li.Buffers(ctx, k, want_scores=True)
    li.forward(ctx, [k], buf)
    torch.cuda.synchronize()
    u16 = lambda t: t.view(torch.int16).numpy().view(np.uint16)
    osel, osc = O.block_select(u16(q), u16(kc), fi, fo, 1, blk, blk, [k])
    np.testing.assert_array_equal(buf.sel_idx.cpu().numpy()[0], osel[0])     # ties are exact: bit-identical mask
    o_ref, lse_ref = O.sparse_attn(u16(q), u16(kc), u16(vc), fi, fo, 1, blk, blk, osel)
    P.compare_output(buf.o, buf.lse, o_ref, lse_ref)


def test_batch_of_64_calls(P):
    """LI_MAX_CALLS independent calls in one launch, each with its own frame list and top-k."""
    spec = W.spec_small(name="small-b64", H=1, d=64, block=64, frame_tokens=64, n_cur_frames=1, n_pages=64 * 6,
                        n_mem=tuple(b % 3 for b in range(64)), n_win=tuple(1 + b % 2 for b in range(64)),
                        density=Fraction(1, 2), pages_per_call=6)
    prob = W.build(spec)
    assert prob.B == 64
    excused, mx, mean = P.full_parity(prob)
    print(f"small-b64: excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_select_reuse_kbar_across_denoising_steps(P):
    """li_block_select_reuse_kbar: the history is static inside a chunk, only Q changes between denoising steps.
    After one full select, a second select with a NEW Q and reuse must equal the oracle run on the new Q."""
    import paper_2605_31158_b200 as li
    spec = W.spec_small(name="small-reuse", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=10,
                        n_mem=(2,), n_win=(3,), density=Fraction(1, 2))
    prob = W.build(spec)
    ctx = P.upload(prob)
    buf = li.Buffers(ctx, prob.kmax, want_scores=True)
    li.li_block_select(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, buf.workspace, buf.scores)
    g = torch.Generator().manual_seed(77)
    prob.q = torch.randn(prob.q.shape, generator=g).to(torch.bfloat16)           # next denoising step: new queries
    ctx.q.copy_(prob.q)
    buf.sel_idx.fill_(-7)
    li.li_block_select(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, buf.workspace, buf.scores, reuse_kbar=True)
    torch.cuda.synchronize()
    osel, osc = P.oracle_select(prob)
    P.check_selection(prob, buf, osel, osc)


@pytest.mark.parametrize("three_d", [False, True])
def test_tail_wave_split_matches_oracle_and_unsplit_run(P, three_d):
    """Few query blocks with long tile lists: li_sparse_attn shares every query block between several CTAs (split of
    the last wave) and merges the partial results with a second launch.  The output must match the
    oracle, and the unsplit run (li_problem.flags = LI_FLAG_NO_SPLIT) up to fp32 rounding of the merge."""
    import paper_2605_31158_b200 as li
    kw = dict(grid=(10, 20), block3d=(4, 8, 4)) if three_d else {}
    spec = W.spec_small(name="small-split", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=3, n_pages=24,
                        n_mem=(6,), n_win=(14,), density=Fraction(1, 1), **kw)
    prob = W.build(spec)
    li.lib().li_reset_launch_count()
    excused, mx, mean = P.full_parity(prob)
    assert li.lib().li_launch_count() == 4, "2 select kernels + attention + merge expected (split not taken?)"
    ctx, buf = P.run_gpu(prob)
    o_split, lse_split = buf.o.float().cpu(), buf.lse.cpu()
    li.lib().li_reset_launch_count()
    ctx, buf = P.run_gpu(prob, flags=li.LI_FLAG_NO_SPLIT)
    assert li.lib().li_launch_count() == 3
    assert (buf.o.float().cpu() - o_split).abs().max() <= 4e-3       # one bf16 ulp of |o| <= 0.5
    assert (buf.lse.cpu() - lse_split).abs().max() <= 1e-5
    print(f"small-split: excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_tail_wave_split_with_text_and_uneven_calls(P):
    """Split query blocks in a batch whose calls differ: long history, no history at all (16 half-tiles
    shared by 5 CTAs: ranges of 3-4), top-k 0; plus a ragged text prefix, so split ranges start inside the text tiles."""
    import paper_2605_31158_b200 as li
    from oracle import li_oracle as O
    spec = W.spec_small(name="small-split-text", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=3, n_pages=72,
                        n_mem=(6, 0, 3), n_win=(14, 0, 9), density=Fraction(1, 1), pages_per_call=24)
    prob = W.build(spec)
    prob.top_k[2] = 0
    Lt = 333
    g = torch.Generator().manual_seed(4242)
    tk = torch.randn((prob.B, spec.H, Lt, spec.d), generator=g).to(torch.bfloat16)
    tv = torch.randn((prob.B, spec.H, Lt, spec.d), generator=g).to(torch.bfloat16)
    ctx = li.Context(prob.q.cuda(), prob.k_cache.cuda(), prob.v_cache.cuda(), torch.from_numpy(prob.frame_idx).cuda(),
                     prob.frame_off, spec.n_cur_frames, spec.block, text_k=tk.cuda(), text_v=tv.cuda())
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
    o_ref, lse_ref = O.sparse_attn(prob.u16(prob.q), prob.u16(prob.k_cache), prob.u16(prob.v_cache), prob.frame_idx,
                                   prob.frame_off, spec.n_cur_frames, spec.block, spec.block, gsel,
                                   text_k=u16(tk), text_v=u16(tv))
    mx, mean = P.compare_output(buf.o, buf.lse, o_ref, lse_ref)
    print(f"small-split-text: max-abs {mx:.3g} mean-abs {mean:.3g}")


def test_whole_step_is_cuda_graph_capturable(P):
    """li_block_select + li_sparse_attn (3 launches with programmatic dependencies, here 4 with the split's merge) issue
    no synchronising call, so a step can be captured once and replayed; the replay must reproduce the eager outputs
    bit for bit, also after the inputs changed in place."""
    import paper_2605_31158_b200 as li
    spec = W.spec_small(name="small-graph", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=3, n_pages=24,
                        n_mem=(6,), n_win=(14,), density=Fraction(1, 2))
    prob = W.build(spec)
    ctx, buf = P.run_gpu(prob, want_scores=False)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        li.forward(ctx, prob.top_k, buf, stream=side)
    for seed in (1, 2):
        g = torch.Generator().manual_seed(seed)
        ctx.q.copy_(torch.randn(prob.q.shape, generator=g).to(torch.bfloat16))    # new queries, same buffers
        li.forward(ctx, prob.top_k, buf)
        torch.cuda.synchronize()
        sel, o, lse = buf.sel_idx.clone(), buf.o.clone(), buf.lse.clone()
        buf.sel_idx.fill_(-9); buf.o.zero_(); buf.lse.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(buf.sel_idx, sel) and torch.equal(buf.o, o) and torch.equal(buf.lse, lse)


def test_calls_on_two_streams_overlap_without_interference(P):
    """include/li.h: calls share no state beyond what the caller passes (own workspace, own outputs).  Two different
    problems are issued alternately on two streams, many times, so that their kernels overlap on the GPU (both grids are
    far below one wave, both take the key-range split and its merge buffers in their OWN workspace); every result must
    equal the one the same call gives when run alone."""
    import paper_2605_31158_b200 as li
    specs = [W.spec_small(name="conc-a", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=3, n_pages=24,
                          n_mem=(6,), n_win=(14,), density=Fraction(1, 2)),
             W.spec_small(name="conc-b", seed=7117, H=3, d=64, block=64, frame_tokens=72, n_cur_frames=3, n_pages=48,
                          n_mem=(12,), n_win=(28,), density=Fraction(1, 3))]
    probs = [W.build(sp) for sp in specs]
    runs = [P.run_gpu(pr, want_scores=False) for pr in probs]          # alone, on the current stream
    refs = [(b.sel_idx.clone(), b.sel_cnt.clone(), b.o.clone(), b.lse.clone()) for _, b in runs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for s_ in streams:
        s_.wait_stream(torch.cuda.current_stream())
    for rep in range(20):
        for (ctx, buf), pr, s_ in zip(runs, probs, streams):
            with torch.cuda.stream(s_):
                buf.sel_idx.fill_(-9)
                buf.o.zero_()
                li.forward(ctx, pr.top_k, buf, stream=s_)
        torch.cuda.synchronize()
        for (ctx, buf), ref in zip(runs, refs):
            assert torch.equal(buf.sel_idx, ref[0]) and torch.equal(buf.sel_cnt, ref[1]), f"rep {rep}: mask differs"
            assert torch.equal(buf.o.view(torch.int16), ref[2].view(torch.int16)), f"rep {rep}: O differs"
            assert torch.equal(buf.lse.view(torch.int32), ref[3].view(torch.int32))


@pytest.mark.parametrize("d,block", [(64, 64), (128, 64), (64, 128)])
def test_tail_wave_split_other_tile_shapes(P, d, block):
    """The split instances of the other (d, block) template variants: 64-key blocks (32-key half-tiles) and d = 64."""
    import paper_2605_31158_b200 as li
    spec = W.spec_small(name=f"small-split-{d}-{block}", H=2, d=d, block=block, frame_tokens=72, n_cur_frames=3, n_pages=48,
                        n_mem=(12,), n_win=(28,), density=Fraction(1, 1))
    prob = W.build(spec)
    li.lib().li_reset_launch_count()
    excused, mx, mean = P.full_parity(prob)
    assert li.lib().li_launch_count() == 4, "split not taken"
    print(f"small-split d={d} block={block}: excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_outputs_are_bitwise_repeatable(P):
    """No atomics on data, fixed reduction orders, every hand-off through mbarriers: repeated runs (also with the
    tail-wave split and its merge) must reproduce mask, O and LSE bit for bit -- a race would show up here."""
    import paper_2605_31158_b200 as li
    spec = W.spec_small(name="small-repeat", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=3, n_pages=24,
                        n_mem=(6,), n_win=(14,), density=Fraction(1, 2))
    prob = W.build(spec)
    ctx, buf = P.run_gpu(prob, want_scores=False)
    ref = (buf.sel_idx.clone(), buf.o.clone(), buf.lse.clone())
    junk = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
    for it in range(20):
        if it % 2:
            junk.fill_(it)                                  # perturb cache state and timing
        buf.sel_idx.fill_(-5); buf.o.fill_(float("nan")); buf.lse.fill_(float("nan"))
        li.forward(ctx, prob.top_k, buf)
        torch.cuda.synchronize()
        assert torch.equal(buf.sel_idx, ref[0]) and torch.equal(buf.o, ref[1]) and torch.equal(buf.lse, ref[2]), it


@pytest.mark.parametrize("T_f,block,d", [(8, 64, 64), (16, 128, 128), (24, 64, 128), (56, 128, 64)])
def test_frames_shorter_than_half_a_block(P, T_f, block, d):
    """frame_tokens < block/2: no tensor map with a half-tile box exists (AttnParams.has_box_full == 0), every K/V
    half-tile is assembled from 8-row TMA boxes out of several pages, and the pool kernel looks a page up per row."""
    spec = W.spec_small(name=f"small-shortframes-{T_f}-{block}", H=2, d=d, block=block, frame_tokens=T_f, n_cur_frames=11,
                        n_pages=64, n_mem=(9,), n_win=(21,), density=Fraction(1, 2))
    prob = W.build(spec)
    assert T_f < block // 2 and prob.M(0) > 2 and prob.L_hist(0) % block != 0
    excused, mx, mean = P.full_parity(prob)
    print(f"{spec.name}: M={prob.M(0)} Nqb={prob.Nqb} excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_caller_built_unsorted_mask(P):
    """li_sparse_attn takes a row of sel_idx as a SET (li.h: distinct values, any order).  A caller-built mask whose rows
    are shuffled -- the partial history tail block M-1 first, in the middle or absent -- must give the oracle's result for
    that set, and li_validate must accept it."""
    import paper_2605_31158_b200 as li
    spec = W.spec_small(name="small-unsorted", H=3, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=14,
                        n_mem=(3,), n_win=(4,), density=Fraction(1, 2))
    prob = W.build(spec)
    M, k = prob.M(0), 6
    assert prob.L_hist(0) % spec.block != 0 and M >= 8            # block M-1 is partial
    rng = np.random.default_rng(31)
    sel = np.full((1, spec.H, prob.Nqb, k), -1, np.int32)
    cnt = np.zeros((1, spec.H, prob.Nqb), np.int32)
    for h in range(spec.H):
        for i in range(prob.Nqb):
            c = int(rng.integers(1, k + 1))
            row = rng.permutation(M - 1)[:c]
            mode = (h + i) % 3                                    # 0: tail block first, 1: somewhere, 2: absent
            if mode == 0:
                row[0] = M - 1
            elif mode == 1:
                row[int(rng.integers(c))] = M - 1
            sel[0, h, i, :c], cnt[0, h, i] = row, c
    ctx = P.upload(prob)
    buf = li.Buffers(ctx, k)
    buf.sel_idx.copy_(torch.from_numpy(sel))
    buf.sel_cnt.copy_(torch.from_numpy(cnt))
    err = torch.full((4,), 7, dtype=torch.int32, device="cuda")
    li.li_validate(ctx, err, buf.sel_idx, buf.sel_cnt, k)
    li.li_sparse_attn(ctx, buf.sel_idx, buf.sel_cnt, k, buf.o, buf.lse, buf.workspace)
    torch.cuda.synchronize()
    assert err.tolist() == [0, 0, 0, 0]
    o_ref, lse_ref = P.oracle_attn(prob, [sel[0]])
    mx, mean = P.compare_output(buf.o, buf.lse, o_ref, lse_ref)
    print(f"small-unsorted: max-abs {mx:.3g} mean-abs {mean:.3g}")


def test_validate_reports_bad_device_inputs(P):
    """li_validate (li.h): page ids outside the pool, sel_cnt > kmax, sel_idx outside [0, M_b), duplicates in a row --
    each found on the device and reported through the caller's error word; a page id outside the pool is never
    dereferenced by li_block_select (its rows count as zeros), so the call after a failed validation cannot fault."""
    import paper_2605_31158_b200 as li
    spec = W.spec_small(name="small-validate", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=16,
                        n_mem=(2, 1), n_win=(3, 2), density=Fraction(1, 2), pages_per_call=8)
    prob = W.build(spec)
    ctx, buf = P.run_gpu(prob, want_scores=False)
    err = torch.full((4,), 7, dtype=torch.int32, device="cuda")

    def check(sel=None, cnt=None):
        li.li_validate(ctx, err, sel, cnt, buf.kmax if sel is not None else 0)
        torch.cuda.synchronize()
        return err.tolist()

    assert check() == [0, 0, 0, 0]
    assert check(buf.sel_idx, buf.sel_cnt) == [0, 0, 0, 0]
    # a page id outside the pool, in call 1's list
    pos = int(prob.frame_off[1]) + 1
    good = int(ctx.frame_idx[pos])
    ctx.frame_idx[pos] = spec.n_pages + 5
    assert check() == [li.LI_BAD_PAGE_ID, 2, pos, spec.n_pages + 5]
    li.li_block_select(ctx, prob.top_k, buf.kmax, buf.sel_idx.clone(), buf.sel_cnt.clone(), buf.workspace)   # must not fault
    torch.cuda.synchronize()
    ctx.frame_idx[pos] = -1
    assert check()[0] == li.LI_BAD_PAGE_ID
    ctx.frame_idx[pos] = good
    # selection lists
    k0 = int(prob.top_k[0])
    assert k0 >= 2
    sel, cnt = buf.sel_idx.clone(), buf.sel_cnt.clone()
    cnt[0, 1, 0] = buf.kmax + 1
    assert check(sel, cnt) == [li.LI_BAD_SEL_CNT, 1, 1 * prob.Nqb + 0, buf.kmax + 1]
    cnt.copy_(buf.sel_cnt)
    sel[1, 0, 1, 0] = prob.M(1)
    assert check(sel, cnt) == [li.LI_BAD_SEL_RANGE, 2, (0 * prob.Nqb + 1) * buf.kmax + 0, prob.M(1)]
    sel.copy_(buf.sel_idx)
    sel[0, 0, 0, 1] = sel[0, 0, 0, 0]
    got = check(sel, cnt)
    assert got[0] == li.LI_BAD_SEL_DUPLICATE and got[1] == 1 and got[2] in (0, 1) and got[3] == int(sel[0, 0, 0, 0])
    sel[0, 0, 0, 0] = -3
    assert check(sel, cnt)[0] == li.LI_BAD_SEL_RANGE
    with pytest.raises(li.LiError):
        li.li_validate(ctx, err, buf.sel_idx, None, buf.kmax)
