"""CPU ORACLE for the Light Interaction AR-aware block-sparse attention path.

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only `tests/`, `__graft_entry__.smoke()`
and the `cpu_baseline` / `--impl reference` legs of `bench.py` may import it.  It shares no
code with the CUDA path (paper_2605_31158_b200/): no kernels, headers, helpers or tables.

It is a plain, slow, step-by-step restatement of PAPER.md section 3.3:
  Eq. 9  block mean pooling of Q and of the historical K, per head;
  Eq. 10  block relevance score  qbar_i . kbar_m / sqrt(d)  and Top_{floor(rM)};
  Eq. 11  attention context  C_i = T  U  K^curr  U  S_i   (T = text, absent here);
  then ordinary scaled-dot-product softmax attention of the query block over C_i
  (PAPER.md:146 names a "LongCat-style 3D block sparse attention kernel" as the core and never
  restates softmax attention; reading c7).
The KV context is "reconstructed" (Fig. 2a) from a frame-paged cache through a
frame-index list  memory | temporal window | current chunk  (BASELINE.json north_star (b)).

Arithmetic: inputs are bf16 bit patterns (uint16) widened EXACTLY, or float arrays used as
they are; every sum, product, exp and division is IEEE fp64 (numpy).  Two places round to
fp32 on purpose, because a floating-point value decides an integer there and both sides must
take that decision in the kernel's precision (fp32): the pooled means and the block scores.
numpy library primitives used as steps: `@` (matmul), `mean`, `exp`, `max`, `sum`, `lexsort`.

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): hand-worked example in
tests/golden/hand_example.json; brute-force dense masked softmax; torch SDPA (library
routine) for r=1 and r->0; rows of exp(s-lse) sum to 1; constant V; shift invariance;
single attended token; page-permutation / duplicate-page / identity-list invariances; pooled
means of constant blocks, ragged tails, NaN padding; closed-form ranking; argsort brute
force; exact ties -> lowest index; k=M; nested selections.
The 3-D block tiling of PAPER.md:129/:321 (functions *_3d at the end) is pinned by tests/test_oracle_3d_pins.py:
explicit coordinate brute force, reduction to the 1-D tiling when blocks are row segments, partition and padding
properties.  The text set T of Eq. 11 (text_k / text_v arguments) is pinned in the same files (brute force, dense SDPA over
[text | context], text-only attention).  Nothing in this file is "parity unpinned".  (The context policy of Eq. 1-4 has
its own oracle, li_policy_oracle.py; Eq. 5-8, the denoising cache, are out of the hot-path scope.)
"""
from __future__ import annotations

import math
from typing import List, Optional, Sequence, Tuple

import numpy as np


# ----------------------------------------------------------------------------- inputs
def widen(x: np.ndarray) -> np.ndarray:
    """bf16 bit patterns (uint16) -> the exact same values in fp64.  Float arrays pass through."""
    x = np.asarray(x)
    if x.dtype == np.uint16:
        return (x.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return x.astype(np.float64)


# ----------------------------------------------------------------------------- step 1
def split_frames(frames_b: Sequence[int], n_cur_frames: int) -> Tuple[List[int], List[int]]:
    """Frame list of one call, logical order memory | window | chunk (north_star):
    the last n_cur_frames entries are the current chunk, the rest is history."""
    frames_b = [int(p) for p in frames_b]
    n_hist = len(frames_b) - n_cur_frames
    assert n_hist >= 0
    return frames_b[:n_hist], frames_b[n_hist:]


def gather_logical(cache: np.ndarray, pages: Sequence[int], h: int) -> np.ndarray:
    """Logical token t of the region lives in page pages[t div T_f] at row t mod T_f.
    cache: [n_pages, H, T_f, d].  Returns fp64 [len(pages)*T_f, d] (empty -> [0, d])."""
    d = cache.shape[-1]
    if len(pages) == 0:
        return np.zeros((0, d), dtype=np.float64)
    return np.concatenate([widen(cache[p, h]) for p in pages], axis=0)


# ----------------------------------------------------------------------------- step 2/3
def block_means(x: np.ndarray, block: int) -> np.ndarray:
    """Eq. 9: mean over the block's VALID tokens (|Q_i|, |K_m| = true count; only
    the last block of a grid may be partial).  x: fp64 [L, d] -> fp32 [ceil(L/block), d]."""
    L, d = x.shape
    n = -(-L // block)
    out = np.zeros((n, d), dtype=np.float32)
    for i in range(n):
        rows = x[i * block: min(L, (i + 1) * block)]
        out[i] = rows.mean(axis=0).astype(np.float32)       # fp64 mean, rounded once to fp32
    return out


# ----------------------------------------------------------------------------- step 4
def block_scores(qbar: np.ndarray, kbar: np.ndarray, d: int) -> np.ndarray:
    """Eq. 10: s_{i,m} = qbar_i . kbar_m / sqrt(d); fp64 from the fp32 pooled
    values, rounded once to fp32.  [Nqb, d] x [M, d] -> fp32 [Nqb, M]."""
    s = (qbar.astype(np.float64) @ kbar.astype(np.float64).T) / math.sqrt(d)
    return s.astype(np.float32)


# ----------------------------------------------------------------------------- step 5
def top_k_rows(scores: np.ndarray, k: int) -> np.ndarray:
    """Top_k of Eq. 10 per row under the total order (score descending, index ascending):
    ties go to the lowest block index (north_star; reading c5).  Returns the chosen
    indices of each row in ASCENDING order, int32 [Nqb, k]."""
    n, M = scores.shape
    k = min(k, M)
    out = np.zeros((n, k), dtype=np.int32)
    idx = np.arange(M)
    for i in range(n):
        order = np.lexsort((idx, -scores[i].astype(np.float64)))   # primary: -score, then index
        out[i] = np.sort(order[:k])
    return out


def block_select(q, k_cache, frame_idx, frame_off, n_cur_frames: int, block_q: int, block_k: int,
                 top_k: Sequence[int]):
    """li_block_select: steps 1-5 for every call b and head h.
    q [B,H,Lq,d]; k_cache [n_pages,H,T_f,d]; frame_idx/frame_off: CSR frame lists; top_k[b].
    Returns per call b: sel_idx int32 [H,Nqb,k_b] (ascending), scores fp32 [H,Nqb,M_b]."""
    B, H, Lq, d = q.shape
    sel, sc = [], []
    for b in range(B):
        hist, _cur = split_frames(frame_idx[frame_off[b]:frame_off[b + 1]], n_cur_frames)
        idx_b, sc_b = [], []
        for h in range(H):
            qbar = block_means(widen(q[b, h]), block_q)
            kbar = block_means(gather_logical(k_cache, hist, h), block_k)
            s = block_scores(qbar, kbar, d)
            M = kbar.shape[0]
            idx_b.append(top_k_rows(s, min(int(top_k[b]), M)))
            sc_b.append(s)
        sel.append(np.stack(idx_b))
        sc.append(np.stack(sc_b))
    return sel, sc


# ----------------------------------------------------------------------------- step 6
def attended_rows(L_hist: int, block_k: int, sel_row: Sequence[int]) -> np.ndarray:
    """Valid logical history tokens of the selected blocks S_i (Eq. 11): block m covers tokens
    [m*Bk, min(L_hist, (m+1)*Bk))."""
    parts = [np.arange(m * block_k, min(L_hist, (m + 1) * block_k)) for m in sel_row]
    return np.concatenate(parts) if parts else np.zeros((0,), dtype=np.int64)


def softmax_attend(qr: np.ndarray, K: np.ndarray, V: np.ndarray, scale: float):
    """o_u = sum_n softmax_n(scale * q_u . k_n) v_n ; lse_u = log sum_n exp(scale * q_u . k_n).
    Two-pass (max, then exp / sum), fp64.  An empty context gives o = 0, lse = -inf."""
    if K.shape[0] == 0:
        return np.zeros((qr.shape[0], V.shape[1])), np.full((qr.shape[0],), -np.inf)
    s = scale * (qr @ K.T)
    mx = s.max(axis=1, keepdims=True)
    e = np.exp(s - mx)
    den = e.sum(axis=1, keepdims=True)
    o = (e @ V) / den
    lse = (mx + np.log(den))[:, 0]
    return o, lse


def sparse_attn(q, k_cache, v_cache, frame_idx, frame_off, n_cur_frames: int, block_q: int,
                block_k: int, sel_idx: Sequence[np.ndarray], softmax_scale: float = 0.0,
                tiles: Optional[Sequence[Tuple[int, int, int]]] = None, text_k=None, text_v=None):
    """li_sparse_attn: step 6 for every (call, head, query block), or only for `tiles`
    = [(b, h, i), ...] (sampled parity at full size).  sel_idx[b]: int [H,Nqb,k_b]; negative
    entries are padding.  Query block i attends ALL chunk tokens (K^curr, no mask inside the
    chunk: DESIGN.md c8) plus the valid tokens of its selected history blocks, plus -- when text_k / text_v
    [B,H,Lt,d] are given -- ALL text-conditioning tokens: C_i = T U K^curr U S_i (Eq. 11, PAPER.md:142-144;
    "the model retains all text-conditioning tokens").
    Returns o fp32 [B,H,Lq,d], lse fp32 [B,H,Lq]  (untouched tiles stay NaN when `tiles`)."""
    B, H, Lq, d = q.shape
    scale = softmax_scale if softmax_scale != 0.0 else 1.0 / math.sqrt(d)
    fill = np.nan if tiles is not None else 0.0
    o = np.full((B, H, Lq, d), fill, dtype=np.float32)
    lse = np.full((B, H, Lq), fill, dtype=np.float32)
    Nqb = -(-Lq // block_q)
    todo = tiles if tiles is not None else [(b, h, i) for b in range(B) for h in range(H) for i in range(Nqb)]
    cache = {}
    for (b, h, i) in todo:
        if (b, h) not in cache:
            cache.clear()
            hist, cur = split_frames(frame_idx[frame_off[b]:frame_off[b + 1]], n_cur_frames)
            cache[(b, h)] = (gather_logical(k_cache, hist, h), gather_logical(v_cache, hist, h),
                             gather_logical(k_cache, cur, h), gather_logical(v_cache, cur, h))
        Kh, Vh, Kc, Vc = cache[(b, h)]
        rows = [int(m) for m in np.asarray(sel_idx[b])[h, i] if int(m) >= 0]
        t = attended_rows(Kh.shape[0], block_k, rows)
        K = np.concatenate([Kc, Kh[t]], axis=0)             # C_i = K^curr U S_i  (Eq. 11)
        V = np.concatenate([Vc, Vh[t]], axis=0)             # same indices for K and V
        if text_k is not None:                              # ... U T: the text tokens are always kept (Eq. 11)
            K = np.concatenate([widen(text_k[b, h]), K], axis=0)
            V = np.concatenate([widen(text_v[b, h]), V], axis=0)
        u0, u1 = i * block_q, min(Lq, (i + 1) * block_q)
        oi, li = softmax_attend(widen(q[b, h, u0:u1]), K, V, scale)
        o[b, h, u0:u1] = oi.astype(np.float32)
        lse[b, h, u0:u1] = li.astype(np.float32)
    return o, lse


# ----------------------------------------------------------------------------- tie report
def excused_mismatch(scores_row: np.ndarray, k: int, got: Sequence[int], want: Sequence[int],
                     rel: float = 1e-4, abs_floor: float = 1e-7) -> bool:
    """north_star: a block-mask disagreement is excused (and reported) iff every block in the
    symmetric difference has an oracle score within rel*|s_(k)| (+abs_floor) of the k-th score."""
    if k <= 0:
        return len(got) == 0
    s = scores_row.astype(np.float64)
    kth = np.sort(s)[::-1][k - 1]
    tol = rel * abs(kth) + abs_floor
    diff = set(int(x) for x in got) ^ set(int(x) for x in want)
    if any(m < 0 or m >= len(s) for m in diff):
        return False
    return all(abs(s[m] - kth) <= tol for m in diff)


# ============================================================================= 3-D block tiling
# "tokens are partitioned into non-overlapping 3D blocks of size (B_t, B_h, B_w)"; (4,8,4) on
# HY-WorldPlay and (4,4,8) on Matrix-Game-3.0, block volume 128 tokens.  A frame is a grid_h x grid_w
# latent grid in row-major token order (token = y*grid_w + x); a region (history or chunk) of n frames in logical
# order is tiled by temporal groups of B_t consecutive frames x B_h rows x B_w columns.  Blocks at the bottom / right
# border and the last temporal group may be partial: "Boundary cases are handled by masked loads",
# "discarding invalid boundary-padding positions through masked stores" -- i.e. padding never counts.
# Block order (reading c17): m = (tg * Hb + hb) * Wb + wb, temporal group slowest.
def blocks_3d(n_frames: int, grid_h: int, grid_w: int, bt: int, bh: int, bw: int) -> List[np.ndarray]:
    """Logical token indices (frame*T_f + y*grid_w + x, ascending) of every 3-D block of a region of n_frames."""
    T_f = grid_h * grid_w
    out = []
    for tg in range(-(-n_frames // bt)):
        for hb in range(-(-grid_h // bh)):
            for wb in range(-(-grid_w // bw)):
                idx = [f * T_f + y * grid_w + x
                       for f in range(tg * bt, min(n_frames, (tg + 1) * bt))
                       for y in range(hb * bh, min(grid_h, (hb + 1) * bh))
                       for x in range(wb * bw, min(grid_w, (wb + 1) * bw))]
                out.append(np.asarray(idx, dtype=np.int64))
    return out


def means_over(x: np.ndarray, blocks: Sequence[np.ndarray]) -> np.ndarray:
    """Eq. 9 over arbitrary token sets: mean of the block's valid tokens, fp64 -> fp32."""
    out = np.zeros((len(blocks), x.shape[1]), dtype=np.float32)
    for i, idx in enumerate(blocks):
        out[i] = x[idx].mean(axis=0).astype(np.float32)
    return out


def block_select_3d(q, k_cache, frame_idx, frame_off, n_cur_frames: int, grid_h: int, grid_w: int, bt: int, bh: int,
                    bw: int, top_k: Sequence[int]):
    """li_block_select with 3-D blocks: same steps as block_select, only the token sets of the blocks differ."""
    B, H, Lq, d = q.shape
    qblocks = blocks_3d(n_cur_frames if n_cur_frames > 0 else Lq // (grid_h * grid_w), grid_h, grid_w, bt, bh, bw)
    sel, sc = [], []
    for b in range(B):
        hist, _cur = split_frames(frame_idx[frame_off[b]:frame_off[b + 1]], n_cur_frames)
        kblocks = blocks_3d(len(hist), grid_h, grid_w, bt, bh, bw)
        idx_b, sc_b = [], []
        for h in range(H):
            qbar = means_over(widen(q[b, h]), qblocks)
            kbar = means_over(gather_logical(k_cache, hist, h), kblocks) if kblocks else np.zeros((0, d), np.float32)
            s = block_scores(qbar, kbar, d)
            idx_b.append(top_k_rows(s, min(int(top_k[b]), len(kblocks))))
            sc_b.append(s)
        sel.append(np.stack(idx_b))
        sc.append(np.stack(sc_b))
    return sel, sc


def sparse_attn_3d(q, k_cache, v_cache, frame_idx, frame_off, n_cur_frames: int, grid_h: int, grid_w: int, bt: int,
                   bh: int, bw: int, sel_idx: Sequence[np.ndarray], softmax_scale: float = 0.0,
                   tiles: Optional[Sequence[Tuple[int, int, int]]] = None, text_k=None, text_v=None):
    """li_sparse_attn with 3-D blocks: the queries of 3-D query block i attend ALL chunk tokens plus the valid tokens
    of the selected 3-D history blocks; outputs in the original linear token order."""
    B, H, Lq, d = q.shape
    scale = softmax_scale if softmax_scale != 0.0 else 1.0 / math.sqrt(d)
    fill = np.nan if tiles is not None else 0.0
    o = np.full((B, H, Lq, d), fill, dtype=np.float32)
    lse = np.full((B, H, Lq), fill, dtype=np.float32)
    qblocks = blocks_3d(n_cur_frames if n_cur_frames > 0 else Lq // (grid_h * grid_w), grid_h, grid_w, bt, bh, bw)
    todo = tiles if tiles is not None else [(b, h, i) for b in range(B) for h in range(H) for i in range(len(qblocks))]
    cache = {}
    for (b, h, i) in todo:
        if (b, h) not in cache:
            cache.clear()
            hist, cur = split_frames(frame_idx[frame_off[b]:frame_off[b + 1]], n_cur_frames)
            cache[(b, h)] = (gather_logical(k_cache, hist, h), gather_logical(v_cache, hist, h),
                             gather_logical(k_cache, cur, h), gather_logical(v_cache, cur, h),
                             blocks_3d(len(hist), grid_h, grid_w, bt, bh, bw))
        Kh, Vh, Kc, Vc, kblocks = cache[(b, h)]
        rows = [int(m) for m in np.asarray(sel_idx[b])[h, i] if int(m) >= 0]
        t = np.concatenate([kblocks[m] for m in rows]) if rows else np.zeros((0,), dtype=np.int64)
        K = np.concatenate([Kc, Kh[t]], axis=0)
        V = np.concatenate([Vc, Vh[t]], axis=0)
        if text_k is not None:                              # T of Eq. 11: always kept
            K = np.concatenate([widen(text_k[b, h]), K], axis=0)
            V = np.concatenate([widen(text_v[b, h]), V], axis=0)
        u = qblocks[i]
        oi, li = softmax_attend(widen(q[b, h])[u], K, V, scale)
        o[b, h, u] = oi.astype(np.float32)
        lse[b, h, u] = li.astype(np.float32)
    return o, lse
