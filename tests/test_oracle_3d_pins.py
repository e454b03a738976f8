"""Pins for the 3-D block tiling of the oracle (oracle/li_oracle.py *_3d), CPU only.  Each test
checks it against something that is not itself: a hand-enumerated example, an independent coordinate-arithmetic brute
force, the 1-D oracle in the case where 3-D blocks degenerate to row segments, torch SDPA for r = 1."""
import math

import numpy as np
import torch

from oracle import li_oracle as O

RNG = np.random.default_rng(31158)


def test_hand_enumerated_blocks():
    """grid 3 x 5, 3 frames, blocks (2,2,2): Hb=2, Wb=3, 2 temporal groups -> 12 blocks.  Token = f*15 + y*5 + x."""
    blocks = O.blocks_3d(3, 3, 5, 2, 2, 2)
    assert len(blocks) == 12
    # block 0: frames 0-1, rows 0-1, cols 0-1
    assert blocks[0].tolist() == [0, 1, 5, 6, 15, 16, 20, 21]
    # block 2: frames 0-1, rows 0-1, col 4 only (right border: 5 = 2+2+1)
    assert blocks[2].tolist() == [4, 9, 19, 24]
    # block 5: frames 0-1, row 2 only (bottom border), col 4 only
    assert blocks[5].tolist() == [14, 29]
    # block 6: second temporal group = frame 2 only (partial group), rows 0-1, cols 0-1
    assert blocks[6].tolist() == [30, 31, 35, 36]
    # block 11: frame 2, row 2, col 4
    assert blocks[11].tolist() == [44]
    # a partition: every token of the region exactly once
    allt = np.sort(np.concatenate(blocks))
    assert allt.tolist() == list(range(45))


def test_paper_geometry_counts():
    """HY-WorldPlay instantiation: 30 x 52 grid, (4,8,4): 4 x 13 = 52 blocks per temporal group, volume 128;
    the bottom row of blocks holds 6 of 8 rows -> 96 tokens."""
    blocks = O.blocks_3d(4, 30, 52, 4, 8, 4)
    assert len(blocks) == 52
    sizes = [len(b) for b in blocks]
    assert sizes[:39] == [128] * 39 and sizes[39:] == [96] * 13 and sum(sizes) == 4 * 1560
    blocks2 = O.blocks_3d(6, 30, 52, 4, 4, 8)            # Matrix-Game geometry, partial temporal group of 2 frames
    assert len(blocks2) == 2 * 8 * 7 and len(blocks2[0]) == 128 and len(blocks2[-1]) == 2 * 2 * 4


def rand_problem(H=2, d=8, gh=3, gw=4, n_pages=9, frames=(5, 1, 4, 2, 6, 8, 0), n_cur=2):
    T_f = gh * gw
    q = RNG.standard_normal((1, H, n_cur * T_f, d))
    kc = RNG.standard_normal((n_pages, H, T_f, d))
    vc = RNG.standard_normal((n_pages, H, T_f, d))
    fi = np.asarray(frames, np.int32)
    fo = np.asarray([0, len(frames)], np.int32)
    return q, kc, vc, fi, fo


def brute_3d(q, kc, vc, frames, n_cur, gh, gw, bt, bh, bw, sel, scale):
    """Independent formulation: block id of a token from coordinate arithmetic, dense masked softmax in loops."""
    H, Lq, d = q.shape
    T_f = gh * gw
    n_hist = len(frames) - n_cur
    Hb, Wb = -(-gh // bh), -(-gw // bw)

    def bid(t):                                   # logical token of a region -> 3-D block id
        f, r = divmod(t, T_f)
        y, x = divmod(r, gw)
        return ((f // bt) * Hb + y // bh) * Wb + x // bw

    out = np.zeros((H, Lq, d)); lse = np.zeros((H, Lq))
    for h in range(H):
        for u in range(Lq):
            allowed = set(int(m) for m in sel[h][bid(u)] if int(m) >= 0)
            logit, val = [], []
            for n in range(n_hist * T_f):
                if bid(n) in allowed:
                    logit.append(scale * float(q[h, u] @ kc[frames[n // T_f], h, n % T_f])); val.append(vc[frames[n // T_f], h, n % T_f])
            for n in range(n_cur * T_f):
                pg = frames[n_hist + n // T_f]
                logit.append(scale * float(q[h, u] @ kc[pg, h, n % T_f])); val.append(vc[pg, h, n % T_f])
            mx = max(logit); w = [math.exp(z - mx) for z in logit]; Z = sum(w)
            out[h, u] = sum(wi * vi for wi, vi in zip(w, val)) / Z
            lse[h, u] = mx + math.log(Z)
    return out, lse


def test_3d_select_and_attention_match_coordinate_brute_force():
    q, kc, vc, fi, fo = rand_problem()
    gh, gw, bt, bh, bw, n_cur = 3, 4, 2, 2, 3, 2          # history 5 frames -> 3 temporal groups (last partial), Hb=2, Wb=2
    M = 3 * 2 * 2
    for k in (0, 1, 5, M):
        sel, sc = O.block_select_3d(q, kc, fi, fo, n_cur, gh, gw, bt, bh, bw, [k])
        assert sc[0].shape == (2, 2 * 2, M)
        # scores straight from the definition: means over explicit coordinate sets
        T_f = gh * gw
        Kh = np.concatenate([kc[p, 0] for p in fi[:5]])
        m = 7                                              # tg=1, hb=1, wb=1: frames 2-3, row 2, col 3
        toks = [f * T_f + 2 * gw + 3 for f in (2, 3)]
        qtok = [f * T_f + y * gw + x for f in (0, 1) for y in (0, 1) for x in (0, 1, 2)]      # query block 0
        want = q[0, 0][qtok].mean(0) @ Kh[toks].mean(0) / math.sqrt(q.shape[-1])
        assert abs(sc[0][0, 0, m] - want) < 1e-5
        o, lse = O.sparse_attn_3d(q, kc, vc, fi, fo, n_cur, gh, gw, bt, bh, bw, sel)
        bo, bl = brute_3d(q[0], kc, vc, list(fi), n_cur, gh, gw, bt, bh, bw, sel[0], 1 / math.sqrt(q.shape[-1]))
        np.testing.assert_allclose(o[0], bo, rtol=1e-5, atol=1e-6)
        np.testing.assert_allclose(lse[0], bl, rtol=1e-5, atol=1e-6)


def test_row_segment_blocks_reduce_to_1d_oracle():
    """(bt,bh,bw) = (1,1,B) with grid_w a multiple of B: 3-D blocks are consecutive runs of B tokens = the 1-D tiling."""
    q, kc, vc, fi, fo = rand_problem(gh=3, gw=4)
    for Bk in (2, 4):
        s3, c3 = O.block_select_3d(q, kc, fi, fo, 2, 3, 4, 1, 1, Bk, [3])
        s1, c1 = O.block_select(q, kc, fi, fo, 2, Bk, Bk, [3])
        np.testing.assert_array_equal(s3[0], s1[0]); np.testing.assert_array_equal(c3[0], c1[0])
        o3, l3 = O.sparse_attn_3d(q, kc, vc, fi, fo, 2, 3, 4, 1, 1, Bk, s3)
        o1, l1 = O.sparse_attn(q, kc, vc, fi, fo, 2, Bk, Bk, s1)
        np.testing.assert_allclose(o3, o1, rtol=1e-6, atol=1e-7); np.testing.assert_allclose(l3, l1, rtol=1e-6, atol=1e-7)


def test_all_blocks_is_dense_and_constant_v():
    q, kc, vc, fi, fo = rand_problem()
    M = 3 * 2 * 2
    sel, _ = O.block_select_3d(q, kc, fi, fo, 2, 3, 4, 2, 2, 3, [M])
    assert (sel[0] == np.arange(M)).all()
    o, _ = O.sparse_attn_3d(q, kc, vc, fi, fo, 2, 3, 4, 2, 2, 3, sel)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a))[None]
    for h in range(2):
        K = np.concatenate([kc[p, h] for p in fi]); V = np.concatenate([vc[p, h] for p in fi])
        ref = torch.nn.functional.scaled_dot_product_attention(t(q[0, h]), t(K), t(V))[0].numpy()
        np.testing.assert_allclose(o[0, h], ref, rtol=1e-5, atol=1e-6)
    c = RNG.standard_normal(q.shape[-1])
    sel2, _ = O.block_select_3d(q, kc, fi, fo, 2, 3, 4, 2, 2, 3, [4])
    o2, _ = O.sparse_attn_3d(q, kc, np.broadcast_to(c, vc.shape).copy(), fi, fo, 2, 3, 4, 2, 2, 3, sel2)
    np.testing.assert_allclose(o2, np.broadcast_to(c, o2.shape), rtol=1e-6, atol=1e-6)


# ----------------------------------------------------------------------------- text prefix T of Eq. 11
def test_text_tokens_are_always_attended():
    """C_i = T U K^curr U S_i: (i) with every block selected the result is dense SDPA over [text | whole context];
    (ii) with no chunk and nothing selected it is SDPA over the text alone; (iii) a brute-force masked softmax in plain
    loops for a partial selection; (iv) K and V of the text are not swapped (V indicator test)."""
    q, kc, vc, fi, fo = rand_problem()
    d = q.shape[-1]
    Lt = 5
    tk = RNG.standard_normal((1, 2, Lt, d)); tv = RNG.standard_normal((1, 2, Lt, d))
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a))[None]
    sdpa = lambda qq, K, V: torch.nn.functional.scaled_dot_product_attention(t(qq), t(K), t(V))[0].numpy()
    # (i) 1-D blocks, everything selected
    Bk = 5
    M = -(-5 * 12 // Bk)
    sel, _ = O.block_select(q, kc, fi, fo, 2, Bk, Bk, [M])
    o, _ = O.sparse_attn(q, kc, vc, fi, fo, 2, Bk, Bk, sel, text_k=tk, text_v=tv)
    for h in range(2):
        K = np.concatenate([tk[0, h]] + [kc[p, h] for p in fi]); V = np.concatenate([tv[0, h]] + [vc[p, h] for p in fi])
        np.testing.assert_allclose(o[0, h], sdpa(q[0, h], K, V), rtol=1e-5, atol=1e-6)
    # (ii) no chunk (n_cur = 0), nothing selected: text only
    o2, _ = O.sparse_attn(q, kc, vc, fi, fo, 0, Bk, Bk, [np.zeros((2, 5, 0), np.int32)], text_k=tk, text_v=tv)
    for h in range(2):
        np.testing.assert_allclose(o2[0, h], sdpa(q[0, h], tk[0, h], tv[0, h]), rtol=1e-5, atol=1e-6)
    # (iii) 3-D blocks, partial selection, brute force in loops
    gh, gw, bt, bh, bw = 3, 4, 2, 2, 3
    sel3, _ = O.block_select_3d(q, kc, fi, fo, 2, gh, gw, bt, bh, bw, [4])
    o3, l3 = O.sparse_attn_3d(q, kc, vc, fi, fo, 2, gh, gw, bt, bh, bw, sel3, text_k=tk, text_v=tv)
    bo, bl = brute_3d(q[0], kc, vc, list(fi), 2, gh, gw, bt, bh, bw, sel3[0], 1 / math.sqrt(d))
    scale = 1 / math.sqrt(d)
    for h in range(2):
        for u in range(q.shape[2]):
            st = scale * (tk[0, h] @ q[0, h, u])
            lse_all = np.logaddexp(bl[h, u], np.log(np.exp(st - st.max()).sum()) + st.max())
            w_ctx = math.exp(bl[h, u] - lse_all)
            want = w_ctx * bo[h, u] + (np.exp(st - lse_all)[:, None] * tv[0, h]).sum(0)
            np.testing.assert_allclose(o3[0, h, u], want, rtol=1e-5, atol=1e-6)
            assert abs(l3[0, h, u] - lse_all) < 1e-5
    # (iv) text K / V roles: only text token 3 matches the query, V is an indicator of the token id
    q1 = np.zeros((1, 1, 12, 4)); q1[..., 0] = 60.0
    tk1 = np.zeros((1, 1, 6, 4)); tk1[0, 0, 3, 0] = 1.0
    tv1 = np.zeros((1, 1, 6, 4)); tv1[0, 0, 3, 2] = 1.0
    z = np.zeros((2, 1, 12, 4))
    o4, _ = O.sparse_attn(q1, z, z, np.asarray([0, 1], np.int32), np.asarray([0, 2], np.int32), 1, 4, 4,
                          [np.zeros((1, 3, 0), np.int32)], text_k=tk1, text_v=tv1)
    assert (o4[0, 0, :, 2] > 0.999).all()
