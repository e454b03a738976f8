"""Shared plumbing of the GPU parity tests: upload a seeded li_workloads.Problem, run the CUDA path through the
C-ABI binding, run the oracle on the same bits, compare.  Holds no arithmetic of the method."""
from __future__ import annotations

import math

import numpy as np
import torch

import li_workloads as W
import paper_2605_31158_b200 as li
from oracle import li_oracle as O

# BASELINE.json north_star: attention output within max-abs 2e-2 and mean-abs 2e-3 of the oracle on bf16 inputs
MAX_ABS, MEAN_ABS = 2e-2, 2e-3
LSE_ABS = 2e-3   # fp32 online softmax vs fp64 two-pass; logits are O(10), ex2.approx/log2 rel. error ~1e-6..1e-7


def upload(prob: W.Problem, dev="cuda:0", flags=0):
    q = prob.q.to(dev)
    kc = prob.k_cache.to(dev)
    vc = prob.v_cache.to(dev)
    fi = torch.from_numpy(prob.frame_idx).to(dev)
    ctx = li.Context(q, kc, vc, fi, prob.frame_off, prob.spec.n_cur_frames, prob.spec.block,
                     grid=prob.spec.grid, block3d=prob.spec.block3d, flags=flags)
    return ctx


def run_gpu(prob: W.Problem, want_scores=True, kmax=None, flags=0):
    ctx = upload(prob, flags=flags)
    buf = li.Buffers(ctx, kmax if kmax is not None else prob.kmax, want_scores=want_scores)
    buf.sel_idx.fill_(-7)
    buf.o.fill_(float("nan"))
    li.forward(ctx, prob.top_k, buf)
    torch.cuda.synchronize()
    return ctx, buf


def gpu_selection(prob: W.Problem, buf):
    """-> per call: sel int32 [H,Nqb,k_b], cnt [H,Nqb], scores [H,Nqb,M_b] (or None)."""
    idx = buf.sel_idx.cpu().numpy()
    cnt = buf.sel_cnt.cpu().numpy()
    sc = buf.scores.cpu().numpy() if buf.scores is not None else None
    out = []
    for b in range(prob.B):
        k = int(prob.top_k[b])
        out.append((idx[b, :, :, :k], cnt[b], sc[b, :, :, :prob.M(b)] if sc is not None else None, idx[b]))
    return out


def check_selection(prob: W.Problem, buf, oracle_sel, oracle_scores):
    """Mask parity: bit-exact, except rows whose symmetric difference lies within the tie window of the k-th
    oracle score (north_star); returns the number of excused rows."""
    excused = 0
    for b, (sel, cnt, sc, raw) in enumerate(gpu_selection(prob, buf)):
        k = int(prob.top_k[b])
        assert (cnt == k).all(), f"sel_cnt mismatch in call {b}"
        assert (raw[:, :, k:] == -1).all(), "entries beyond k must be -1"
        if k > 1:
            assert (np.diff(sel, axis=-1) > 0).all(), "indices must be strictly ascending"
        want = oracle_sel[b]
        if sc is not None:
            np.testing.assert_allclose(sc, oracle_scores[b], rtol=2e-5, atol=2e-6)
        bad = np.argwhere((sel != want).any(axis=-1))
        for h, i in bad:
            assert O.excused_mismatch(oracle_scores[b][h, i], k, sel[h, i], want[h, i]), \
                f"block mask differs outside the tie window: call {b} head {h} row {i}: {sel[h, i]} vs {want[h, i]}"
            excused += 1
    return excused


def oracle_select(prob: W.Problem):
    s = prob.spec
    if s.block3d is not None:
        return O.block_select_3d(prob.u16(prob.q), prob.u16(prob.k_cache), prob.frame_idx, prob.frame_off,
                                 s.n_cur_frames, *s.grid, *s.block3d, prob.top_k)
    return O.block_select(prob.u16(prob.q), prob.u16(prob.k_cache), prob.frame_idx, prob.frame_off,
                          s.n_cur_frames, s.block, s.block, prob.top_k)


def oracle_attn(prob: W.Problem, sel_per_call, tiles=None):
    s = prob.spec
    if s.block3d is not None:
        return O.sparse_attn_3d(prob.u16(prob.q), prob.u16(prob.k_cache), prob.u16(prob.v_cache), prob.frame_idx,
                                prob.frame_off, s.n_cur_frames, *s.grid, *s.block3d, sel_per_call, tiles=tiles)
    return O.sparse_attn(prob.u16(prob.q), prob.u16(prob.k_cache), prob.u16(prob.v_cache), prob.frame_idx,
                         prob.frame_off, s.n_cur_frames, s.block, s.block, sel_per_call, tiles=tiles)


def compare_output(o_gpu: torch.Tensor, lse_gpu, o_ref: np.ndarray, lse_ref: np.ndarray, mask=None):
    og = o_gpu.float().cpu().numpy()
    if mask is not None:
        og, o_ref = og[mask], o_ref[mask]
    assert np.isfinite(og).all(), "non-finite values in O"
    diff = np.abs(og - o_ref)
    assert diff.max() <= MAX_ABS, f"max-abs {diff.max():.4g} > {MAX_ABS}"
    assert diff.mean() <= MEAN_ABS, f"mean-abs {diff.mean():.4g} > {MEAN_ABS}"
    if lse_gpu is not None:
        lg = lse_gpu.cpu().numpy()
        if mask is not None:
            lg, lse_ref = lg[mask], lse_ref[mask]
        assert np.abs(lg - lse_ref).max() <= LSE_ABS, f"lse max-abs {np.abs(lg - lse_ref).max():.4g}"
    return float(diff.max()), float(diff.mean())


def select_parity(prob: W.Problem):
    """Mask + score parity of li_block_select alone."""
    ctx = upload(prob)
    buf = li.Buffers(ctx, prob.kmax, want_scores=True)
    buf.sel_idx.fill_(-7)
    li.li_block_select(ctx, prob.top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, buf.workspace, buf.scores)
    torch.cuda.synchronize()
    osel, osc = oracle_select(prob)
    return check_selection(prob, buf, osel, osc)


def full_parity(prob: W.Problem):
    """Element-by-element parity of select + attention for a problem the oracle finishes in seconds."""
    ctx, buf = run_gpu(prob)
    osel, osc = oracle_select(prob)
    excused = check_selection(prob, buf, osel, osc)
    gsel = [g[0] for g in gpu_selection(prob, buf)]
    o_ref, lse_ref = oracle_attn(prob, gsel)          # oracle attention on the GPU's (validated) mask
    mx, mean = compare_output(buf.o, buf.lse, o_ref, lse_ref)
    return excused, mx, mean
