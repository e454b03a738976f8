"""Pins for oracle/li_oracle.py (CPU only).  Each test checks the oracle against something that is
NOT the oracle: the hand-worked example in tests/golden/, brute force, a library routine (torch
SDPA), closed forms or invariants that PAPER.md Eq. 9-11 and softmax attention fix.  A dropped
term, wrong sign/index or transposed operand in the oracle fails at least one of them."""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

from oracle import li_oracle as O

HERE = os.path.dirname(os.path.abspath(__file__))
RNG = np.random.default_rng(20260531)


# --------------------------------------------------------------------------------------
# helpers (independent of the oracle)
# --------------------------------------------------------------------------------------
def brute_dense_masked(q, k_cache, v_cache, frames, n_cur, Bq, Bk, sel, scale):
    """Independent formulation: build the FULL logical context [history | chunk], a dense
    [Lq, Lk] logit matrix, put -inf wherever Eq. 11 does not attend, and softmax row by row in
    pure Python.  Tiny inputs only."""
    H, Lq, d = q.shape
    T_f = k_cache.shape[2]
    n_hist = len(frames) - n_cur
    L_hist = n_hist * T_f
    Lk = L_hist + n_cur * T_f
    out = np.zeros((H, Lq, d))
    lse = np.zeros((H, Lq))
    for h in range(H):
        for u in range(Lq):
            i = u // Bq
            allowed = set(int(m) for m in sel[h][i] if int(m) >= 0)
            logits, vals = [], []
            for n in range(Lk):
                page = frames[n // T_f]
                row = n % T_f
                if n < L_hist and (n // Bk) not in allowed:
                    continue                                     # -inf
                kv = k_cache[page, h, row]
                logits.append(scale * float(sum(float(q[h, u, c]) * float(kv[c]) for c in range(d))))
                vals.append(v_cache[page, h, row])
            mx = max(logits)
            w = [math.exp(x - mx) for x in logits]
            z = sum(w)
            out[h, u] = sum(wi * np.asarray(vi, dtype=np.float64) for wi, vi in zip(w, vals)) / z
            lse[h, u] = mx + math.log(z)
    return out, lse


def rand_problem(H=2, d=8, T_f=12, n_pages=7, frames=(5, 1, 4, 2, 6), n_cur=2, B=1):
    q = RNG.standard_normal((B, H, n_cur * T_f, d))
    kc = RNG.standard_normal((n_pages, H, T_f, d))
    vc = RNG.standard_normal((n_pages, H, T_f, d))
    fi = np.asarray(list(frames) * B, dtype=np.int32)
    fo = np.arange(B + 1, dtype=np.int32) * len(frames)
    return q, kc, vc, fi, fo


# --------------------------------------------------------------------------------------
# golden: the hand-worked example (Eq. 9-11)
# --------------------------------------------------------------------------------------
def load_hand():
    with open(os.path.join(HERE, "golden", "hand_example.json")) as f:
        g = json.load(f)
    a = math.log(2.0)
    q = np.asarray(g["q_in_units_of_ln2"], dtype=np.float64)[None, None] * a
    kc = np.stack([np.asarray(g["k_pages"][str(p)], dtype=np.float64) for p in range(4)])[:, None]
    vc = np.stack([np.asarray(g["v_pages"][str(p)], dtype=np.float64) for p in range(4)])[:, None]
    fi = np.asarray(g["frames"], dtype=np.int32)
    fo = np.asarray([0, len(fi)], dtype=np.int32)
    return g, q, kc, vc, fi, fo


def test_golden_hand_example_pooling_scores_topk():
    g, q, kc, vc, fi, fo = load_hand()
    a = math.log(2.0)
    hist, cur = O.split_frames(fi, g["n_cur_frames"])
    assert hist == [2, 0] and cur == [3]
    kbar = O.block_means(O.gather_logical(kc, hist, 0), g["block"])
    np.testing.assert_array_equal(kbar, np.asarray(g["expect"]["kbar"], dtype=np.float32))
    qbar = O.block_means(O.widen(q[0, 0]), g["block"])
    np.testing.assert_allclose(qbar / a, np.asarray(g["expect"]["qbar_in_units_of_ln2"]), rtol=1e-6)
    for k, key in ((1, "top1"), (2, "top2"), (3, "top3")):
        sel, sc = O.block_select(q, kc, fi, fo, g["n_cur_frames"], g["block"], g["block"], [k])
        np.testing.assert_array_equal(sel[0][0], np.asarray(g["expect"][key], dtype=np.int32))
        np.testing.assert_allclose(sc[0][0] * math.sqrt(2.0) / a,
                                   np.asarray(g["expect"]["scores_times_sqrt2_over_ln2"]), rtol=1e-6, atol=1e-7)


def test_golden_hand_example_attention():
    g, q, kc, vc, fi, fo = load_hand()
    sel = [np.asarray(g["expect"]["top2"], dtype=np.int32)[None]]
    o, lse = O.sparse_attn(q, kc, vc, fi, fo, g["n_cur_frames"], g["block"], g["block"], sel, softmax_scale=1.0)
    want = np.asarray([[float(Fraction(x)) for x in row] for row in g["expect"]["o_top2"]])
    np.testing.assert_allclose(o[0, 0], want, rtol=1e-6)
    np.testing.assert_allclose(np.exp(lse[0, 0].astype(np.float64)), g["expect"]["exp_lse_top2"], rtol=1e-6)


# --------------------------------------------------------------------------------------
# attention (step 6)
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [0, 1, 2, 4])
def test_attention_equals_bruteforce_dense_masked(k):
    q, kc, vc, fi, fo = rand_problem()
    Bq = Bk = 5                      # 36 history tokens -> M=8 with a ragged tail of 1; Lq=24 -> tail 4
    sel, _ = O.block_select(q, kc, fi, fo, 2, Bq, Bk, [k])
    o, lse = O.sparse_attn(q, kc, vc, fi, fo, 2, Bq, Bk, sel)
    bo, bl = brute_dense_masked(q[0], kc, vc, list(fi), 2, Bq, Bk, sel[0], 1.0 / math.sqrt(q.shape[-1]))
    np.testing.assert_allclose(o[0], bo, rtol=1e-5, atol=1e-6)
    np.testing.assert_allclose(lse[0], bl, rtol=1e-5, atol=1e-6)


def sdpa(qh, K, V, scale):
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a))[None]
    return torch.nn.functional.scaled_dot_product_attention(t(qh), t(K), t(V), scale=scale)[0].numpy()


def test_all_blocks_selected_equals_dense_sdpa():
    """r = 1 (warm-up = 'full dense computation'): library dense attention over the
    gathered context [chunk | history] (softmax is permutation invariant over keys)."""
    q, kc, vc, fi, fo = rand_problem()
    Bq = Bk = 5
    M = -(-36 // Bk)
    sel, _ = O.block_select(q, kc, fi, fo, 2, Bq, Bk, [M])
    assert sel[0].shape[-1] == M and (sel[0] == np.arange(M)).all()          # k = M -> identity set
    o, _ = O.sparse_attn(q, kc, vc, fi, fo, 2, Bq, Bk, sel)
    for h in range(q.shape[1]):
        K = np.concatenate([kc[p, h] for p in fi])
        V = np.concatenate([vc[p, h] for p in fi])
        np.testing.assert_allclose(o[0, h], sdpa(q[0, h], K, V, 1 / math.sqrt(q.shape[-1])), rtol=1e-5, atol=1e-6)


def test_r_to_zero_is_chunk_self_attention():
    """Eq. 11 with S_i empty: C_i = K^curr -> plain bidirectional self-attention of the chunk."""
    q, kc, vc, fi, fo = rand_problem()
    sel, _ = O.block_select(q, kc, fi, fo, 2, 5, 5, [0])
    o, _ = O.sparse_attn(q, kc, vc, fi, fo, 2, 5, 5, sel)
    for h in range(q.shape[1]):
        K = np.concatenate([kc[p, h] for p in fi[-2:]])
        V = np.concatenate([vc[p, h] for p in fi[-2:]])
        np.testing.assert_allclose(o[0, h], sdpa(q[0, h], K, V, 1 / math.sqrt(q.shape[-1])), rtol=1e-5, atol=1e-6)


def test_softmax_rows_sum_to_one_via_lse():
    q, kc, vc, fi, fo = rand_problem()
    Bq = Bk = 5
    sel, _ = O.block_select(q, kc, fi, fo, 2, Bq, Bk, [3])
    _, lse = O.sparse_attn(q, kc, vc, fi, fo, 2, Bq, Bk, sel)
    scale = 1 / math.sqrt(q.shape[-1])
    for h in range(2):
        Kh = np.concatenate([kc[p, h] for p in fi[:3]])
        Kc = np.concatenate([kc[p, h] for p in fi[3:]])
        for u in range(q.shape[2]):
            t = O.attended_rows(Kh.shape[0], Bk, sel[0][h, u // Bq])
            s = scale * (np.concatenate([Kc, Kh[t]]) @ q[0, h, u])
            assert abs(np.exp(s - float(lse[0, h, u])).sum() - 1.0) < 1e-5


def test_constant_v_gives_constant_output_and_single_token():
    q, kc, vc, fi, fo = rand_problem()
    c = RNG.standard_normal(q.shape[-1])
    vconst = np.broadcast_to(c, vc.shape).copy()
    sel, _ = O.block_select(q, kc, fi, fo, 2, 5, 5, [2])
    o, _ = O.sparse_attn(q, kc, vconst, fi, fo, 2, 5, 5, sel)
    np.testing.assert_allclose(o, np.broadcast_to(c, o.shape), rtol=1e-6, atol=1e-6)
    # single attended token: no chunk (n_cur=0), history of one frame with T_f=1, k=1 -> O = that V row
    q1 = RNG.standard_normal((1, 1, 3, 4))
    k1 = RNG.standard_normal((2, 1, 1, 4))
    v1 = RNG.standard_normal((2, 1, 1, 4))
    o1, _ = O.sparse_attn(q1, k1, v1, np.asarray([1], np.int32), np.asarray([0, 1], np.int32), 0, 3, 1,
                          [np.zeros((1, 1, 1), np.int32)])
    np.testing.assert_allclose(o1[0, 0], np.broadcast_to(v1[1, 0, 0], (3, 4)), rtol=1e-6)


def test_shift_invariance_of_selection_and_output():
    """Adding one vector delta to every K row adds a per-row constant to all logits and to all
    block scores of a row: selection and output must not move (exact-arithmetic property)."""
    q, kc, vc, fi, fo = rand_problem()
    delta = RNG.standard_normal(q.shape[-1])
    sel0, _ = O.block_select(q, kc, fi, fo, 2, 5, 5, [3])
    sel1, _ = O.block_select(q, kc + delta, fi, fo, 2, 5, 5, [3])
    np.testing.assert_array_equal(sel0[0], sel1[0])
    o0, _ = O.sparse_attn(q, kc, vc, fi, fo, 2, 5, 5, sel0)
    o1, _ = O.sparse_attn(q, kc + delta, vc, fi, fo, 2, 5, 5, sel0)
    np.testing.assert_allclose(o0, o1, rtol=1e-5, atol=1e-5)


def test_k_and_v_not_swapped_or_transposed():
    """Asymmetric case: K carries all the signal, V is an indicator of the token id; the output's
    argmax must name the key with the largest logit."""
    d, T_f = 6, 6
    q = np.zeros((1, 1, T_f, d)); q[0, 0, :, 0] = 50.0
    kc = np.zeros((2, 1, T_f, d)); vc = np.zeros((2, 1, T_f, d))
    kc[1, 0, 4, 0] = 1.0                       # history page 1, token 4 is the only match
    for t in range(T_f):
        vc[1, 0, t, t] = 1.0
    o, _ = O.sparse_attn(q, kc, vc, np.asarray([1, 0], np.int32), np.asarray([0, 2], np.int32), 1, 6, 6,
                         [np.zeros((1, 1, 1), np.int32)])
    assert (o[0, 0].argmax(axis=1) == 4).all() and (o[0, 0, :, 4] > 0.999).all()


# --------------------------------------------------------------------------------------
# gather (step 1)
# --------------------------------------------------------------------------------------
def test_page_permutation_duplicates_and_identity_list():
    q, kc, vc, fi, fo = rand_problem()
    sel, sc = O.block_select(q, kc, fi, fo, 2, 5, 5, [3])
    o, _ = O.sparse_attn(q, kc, vc, fi, fo, 2, 5, 5, sel)
    # permute the pool and rewrite the list: bit-identical results
    perm = RNG.permutation(kc.shape[0])
    inv = np.argsort(perm)
    sel_p, sc_p = O.block_select(q, kc[perm], inv[fi].astype(np.int32), fo, 2, 5, 5, [3])
    o_p, _ = O.sparse_attn(q, kc[perm], vc[perm], inv[fi].astype(np.int32), fo, 2, 5, 5, sel_p)
    np.testing.assert_array_equal(sel[0], sel_p[0]); np.testing.assert_array_equal(sc[0], sc_p[0])
    np.testing.assert_array_equal(o, o_p)
    # a duplicated page id == a physically duplicated frame
    fd = np.asarray([5, 5, 4, 2, 6], np.int32)
    kc2 = np.concatenate([kc, kc[5:6]]); vc2 = np.concatenate([vc, vc[5:6]])
    fphys = np.asarray([5, 7, 4, 2, 6], np.int32)
    sa, _ = O.block_select(q, kc, fd, fo, 2, 5, 5, [3]); sb, _ = O.block_select(q, kc2, fphys, fo, 2, 5, 5, [3])
    np.testing.assert_array_equal(sa[0], sb[0])
    np.testing.assert_array_equal(O.sparse_attn(q, kc, vc, fd, fo, 2, 5, 5, sa)[0],
                                  O.sparse_attn(q, kc2, vc2, fphys, fo, 2, 5, 5, sb)[0])
    # identity list on a contiguous cache == un-paged attention over [chunk | history] with all blocks
    ident = np.arange(5, dtype=np.int32)
    sel_all = [np.broadcast_to(np.arange(8, dtype=np.int32), (2, 5, 8)).copy()]
    o_id, _ = O.sparse_attn(q, kc, vc, ident, fo, 2, 5, 5, sel_all)
    for h in range(2):
        K = kc[:5, h].reshape(-1, kc.shape[-1]); V = vc[:5, h].reshape(-1, vc.shape[-1])
        np.testing.assert_allclose(o_id[0, h], sdpa(q[0, h], K, V, 1 / math.sqrt(q.shape[-1])), rtol=1e-5, atol=1e-6)


def test_wrong_page_changes_answer():
    q, kc, vc, fi, fo = rand_problem()
    sel, _ = O.block_select(q, kc, fi, fo, 2, 5, 5, [8])
    o, _ = O.sparse_attn(q, kc, vc, fi, fo, 2, 5, 5, sel)
    f2 = fi.copy(); f2[0] = 0
    o2, _ = O.sparse_attn(q, kc, vc, f2, fo, 2, 5, 5, sel)
    assert np.abs(o - o2).max() > 1e-3


# --------------------------------------------------------------------------------------
# pooling (steps 2-3, Eq. 9)
# --------------------------------------------------------------------------------------
def test_block_means_constant_blocks_ragged_tail_and_nan_padding():
    d, Bk = 4, 5
    consts = RNG.standard_normal((4, d)).astype(np.float32).astype(np.float64)
    x = np.repeat(consts, Bk, axis=0)[:17]                 # 17 tokens: blocks 5,5,5,2
    np.testing.assert_array_equal(O.block_means(x, Bk), consts.astype(np.float32))
    y = RNG.standard_normal((17, d))
    m = O.block_means(y, Bk)
    np.testing.assert_allclose(m[3], y[15:17].mean(axis=0), rtol=1e-6)       # true count 2, not 5
    np.testing.assert_allclose(m[1], y[5:10].sum(axis=0) / 5.0, rtol=1e-6)
    # padding never enters a mean: a pool whose other pages are NaN must not propagate
    kc = np.full((3, 1, 6, d), np.nan); kc[1] = RNG.standard_normal((1, 6, d)); kc[2] = RNG.standard_normal((1, 6, d))
    q = RNG.standard_normal((1, 1, 6, d))
    sel, sc = O.block_select(q, kc, np.asarray([1, 2], np.int32), np.asarray([0, 2], np.int32), 1, 4, 4, [1])
    assert np.isfinite(sc[0]).all()


def test_bf16_widening_is_exact():
    t = torch.randn(1000, dtype=torch.float32).to(torch.bfloat16)
    u = t.view(torch.int16).numpy().view(np.uint16)
    np.testing.assert_array_equal(O.widen(u), t.to(torch.float64).numpy())


# --------------------------------------------------------------------------------------
# scores / top-k (steps 4-5, Eq. 10)
# --------------------------------------------------------------------------------------
def test_closed_form_ranking():
    """K block m == c_m * u everywhere, Q == u everywhere: score_m = c_m |u|^2 / sqrt(d), so the
    ranking is the ranking of c_m."""
    d, T_f, Bk = 8, 8, 4
    u = RNG.standard_normal(d)
    c = np.asarray([0.3, -1.0, 2.5, 0.1, 1.7, -0.2])       # 6 blocks = 3 history frames of 8 tokens
    kc = np.zeros((4, 1, T_f, d))
    for m, cm in enumerate(c):
        kc[m // 2, 0, (m % 2) * Bk:(m % 2 + 1) * Bk] = cm * u
    q = np.broadcast_to(u, (1, 1, T_f, d)).copy()
    fi = np.asarray([0, 1, 2, 3], np.int32); fo = np.asarray([0, 4], np.int32)
    for k in range(1, 7):
        sel, sc = O.block_select(q, kc, fi, fo, 1, Bk, Bk, [k])
        want = np.sort(np.argsort(-c)[:k])
        for i in range(2):
            np.testing.assert_array_equal(sel[0][0, i], want)
    np.testing.assert_allclose(sc[0][0, 0], c * (u @ u) / math.sqrt(d), rtol=1e-5)


def test_topk_matches_bruteforce_argsort_and_is_nested():
    q, kc, vc, fi, fo = rand_problem(H=3, d=16, T_f=20, frames=(5, 1, 4, 2, 6, 3, 0), n_cur=2)
    Bk = 7
    prev = None
    for k in range(0, 16):
        sel, sc = O.block_select(q, kc, fi, fo, 2, Bk, Bk, [k])
        M = sc[0].shape[-1]
        assert M == -(-100 // Bk)
        # brute force from raw definitions, straight from the inputs
        for h in range(3):
            Kh = np.concatenate([kc[p, h] for p in fi[:5]])
            for i in range(sel[0].shape[1]):
                qb = q[0, h, i * Bk:(i + 1) * Bk].mean(axis=0)
                s = np.asarray([qb @ Kh[m * Bk:(m + 1) * Bk].mean(axis=0) / math.sqrt(16) for m in range(M)])
                want = set(np.argsort(-s, kind="stable")[:min(k, M)].tolist())
                assert set(sel[0][h, i].tolist()) == want
                assert list(sel[0][h, i]) == sorted(sel[0][h, i])
        if prev is not None:
            for h in range(3):
                for i in range(sel[0].shape[1]):
                    assert set(prev[h, i].tolist()) <= set(sel[0][h, i].tolist())   # I_i(k) subset I_i(k+1)
        prev = sel[0]


def test_exact_ties_pick_lowest_index():
    """Duplicate page ids give bit-identical pooled blocks -> exact score ties."""
    d, T_f, Bk = 8, 8, 8
    kc = RNG.standard_normal((3, 1, T_f, d)); q = RNG.standard_normal((1, 1, T_f, d))
    fi = np.asarray([1, 0, 1, 0, 1, 2], np.int32); fo = np.asarray([0, 6], np.int32)     # history 1,0,1,0,1
    sel, sc = O.block_select(q, kc, fi, fo, 1, Bk, Bk, [1])
    s = sc[0][0, 0]
    assert s[0] == s[2] == s[4] and s[1] == s[3]
    assert sel[0][0, 0, 0] == (0 if s[0] >= s[1] else 1)
    sel2, _ = O.block_select(q, kc, fi, fo, 1, Bk, Bk, [2])
    assert list(sel2[0][0, 0]) == ([0, 2] if s[0] >= s[1] else [1, 3])
    # direct: top_k_rows on a constructed tie
    np.testing.assert_array_equal(O.top_k_rows(np.asarray([[1.0, 3.0, 3.0, 0.0, 3.0]], np.float32), 2), [[1, 2]])
    np.testing.assert_array_equal(O.top_k_rows(np.asarray([[1.0, 3.0, 3.0, 0.0, 3.0]], np.float32), 4), [[0, 1, 2, 4]])


def test_excused_mismatch_rule():
    s = np.asarray([1.0, 0.5, 0.50000001, 0.1], np.float32)
    assert O.excused_mismatch(s, 2, [0, 2], [0, 1])          # swap inside the tie window
    assert not O.excused_mismatch(s, 2, [0, 3], [0, 1])      # 0.1 is nowhere near the k-th score
    assert O.excused_mismatch(s, 2, [0, 1], [0, 1])
