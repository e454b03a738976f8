"""li_block_select_static (include/li.h): the entry point that allocates nothing -- its scratch is a file-scope __device__
array of LI_STATIC_SCRATCH_BYTES inside libli.so.  Collected last on purpose (the suite runs with pytest -x).

The GPU test runs calls IN A ROW on problems of different shape through the shared array (which keeps the previous call's
contents) and checks every output against the existing li_block_select path with a caller workspace: block mask, counts
and scores bit for bit (the bar of tests/test_gpu_parity.py for integer / index work; the two paths run the same kernels
on the same inputs, so the fp32 scores are identical too), and li_sparse_attn on the two masks bit for bit."""
import ctypes
from fractions import Fraction

import numpy as np
import pytest
import torch

import li_workloads as W
import paper_2605_31158_b200 as li


def _fake_problem(**over):
    """A structurally valid li_problem with fake (aligned, never dereferenced) device addresses."""
    fo = np.asarray([0, 4], dtype=np.int32)
    p = li.li_problem()
    p.B, p.H, p.Lq, p.d = 1, 2, 256, 64
    p.frame_tokens, p.block_q, p.block_k, p.n_pages = 256, 64, 64, 8
    p.q = 0x10000
    p.q_sb, p.q_sh, p.q_st = 2 * 256 * 64, 256 * 64, 64
    p.k_cache, p.v_cache = 0x20000, 0x30000
    p.kv_sp, p.kv_sh, p.kv_st = 2 * 256 * 64, 256 * 64, 64
    p.frame_idx = 0x40000
    p.frame_off_host = fo.ctypes.data
    p.n_cur_frames = 1
    p.softmax_scale = 0.0
    for k, v in over.items():
        setattr(p, k, v)
    return p, fo


def test_sizes_beyond_the_static_scratch_are_rejected_before_any_device_work():
    """No GPU needed: the size check comes before the first CUDA call."""
    L = li.lib()
    tk = np.asarray([8], dtype=np.int32)
    p, fo = _fake_problem()
    # qbar [1,2,4,64] fp32 + kbar [1,2,64,32] fp32 + score keys [1,2,4,12] u32 rounded up to 256 B
    assert L.li_static_scratch_needed(ctypes.byref(p)) == 2 * 4 * 64 * 4 + 2 * 64 * 32 * 4 + 512
    assert li.LI_STATIC_SCRATCH_BYTES == 16 << 20
    # 2048 heads of the same shape: 2048 * (1024 + 8192) + keys > 16 MiB
    H = 2048
    big, fo2 = _fake_problem(H=H, q_sb=H * 256 * 64, kv_sp=H * 256 * 64)
    need = L.li_static_scratch_needed(ctypes.byref(big))
    assert need > li.LI_STATIC_SCRATCH_BYTES
    rc = L.li_block_select_static(ctypes.byref(big), tk.ctypes.data, 8, 0x60000, 0x70000, None, 0, None)
    assert rc == li.LI_ERR_TOO_LARGE
    assert "LI_STATIC_SCRATCH_BYTES" in li.strerror(rc)
    # argument checks are those of li_block_select
    assert L.li_block_select_static(None, tk.ctypes.data, 8, 0x60000, 0x70000, None, 0, None) == li.LI_ERR_INVALID_ARG
    bad, fo3 = _fake_problem(d=96)
    assert L.li_block_select_static(ctypes.byref(bad), tk.ctypes.data, 8, 0x60000, 0x70000, None, 0, None) == li.LI_ERR_UNSUPPORTED
    assert L.li_static_scratch_needed(ctypes.byref(bad)) == 0


def _problems():
    """Different shapes one after the other, the largest first, so that every later call finds the array full of another
    problem's pooled means: d = 128 varlen batch (4 calls), the d = 64 `tiny` config, a 3-D tiling, then M > 512 (the
    two-kernel fallback, whose score keys also live in the scratch)."""
    from tests import parity_util as P
    out = []
    spec = W.spec_small(name="noalloc-batch", H=3, d=128, block=128, frame_tokens=200, n_cur_frames=2, n_pages=40,
                        n_mem=(0, 2, 0, 3), n_win=(1, 2, 4, 1), density=Fraction(3, 10), pages_per_call=10)
    prob = W.build(spec)
    out.append((P.upload(prob), list(prob.top_k), prob.kmax))
    prob = W.build(W.spec_tiny())
    out.append((P.upload(prob), list(prob.top_k), prob.kmax))
    spec = W.spec_small(name="noalloc-3d", H=2, d=128, block=64, frame_tokens=10 * 12, n_cur_frames=2, n_pages=14,
                        n_mem=(2,), n_win=(6,), density=Fraction(1, 2), grid=(10, 12), block3d=(2, 4, 8))
    prob = W.build(spec)
    out.append((P.upload(prob), list(prob.top_k), prob.kmax))
    g = torch.Generator().manual_seed(12)
    H, d, T_f, blk, n_hist, k = 1, 64, 64, 64, 700, 600
    q = torch.randn((1, H, T_f, d), generator=g).to(torch.bfloat16)
    kc = torch.randn((7, H, T_f, d), generator=g).to(torch.bfloat16)
    vc = torch.randn((7, H, T_f, d), generator=g).to(torch.bfloat16)
    fi = np.concatenate([torch.randint(0, 6, (n_hist,), generator=g).numpy(), [6]]).astype(np.int32)
    fo = np.asarray([0, n_hist + 1], np.int32)
    out.append((li.Context(q.cuda(), kc.cuda(), vc.cuda(), torch.from_numpy(fi).cuda(), fo, 1, blk), [k], k))
    return out


@pytest.mark.gpu
def test_static_scratch_path_matches_the_workspace_path_on_calls_in_a_row():
    torch.cuda.set_device(0)
    problems = _problems()
    refs = []
    for ctx, top_k, kmax in problems:                      # the existing path, each with its own workspace
        buf = li.Buffers(ctx, kmax, want_scores=True)
        buf.scores.fill_(float("nan"))
        li.forward(ctx, top_k, buf)
        refs.append(buf)
    torch.cuda.synchronize()
    outs = []
    for ctx, top_k, kmax in problems:                      # output tensors made up front: nothing is allocated below
        assert 0 < li.li_static_scratch_needed(ctx) <= li.LI_STATIC_SCRATCH_BYTES
        buf = li.Buffers(ctx, kmax, want_scores=True)
        outs.append(buf)
    li.li_block_select_static(*problems[0][:3], outs[0].sel_idx, outs[0].sel_cnt, outs[0].scores)   # loads the module
    torch.cuda.synchronize()
    launches_before = li.launch_count()
    for rep in range(2):                                   # the whole sequence twice, back to back on one stream
        for buf in outs:
            buf.sel_idx.fill_(-7)
            buf.sel_cnt.fill_(-7)
            buf.scores.fill_(float("nan"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]         # no torch op between the two readings
        for (ctx, top_k, kmax), buf in zip(problems, outs):
            li.li_block_select_static(ctx, top_k, kmax, buf.sel_idx, buf.sel_cnt, buf.scores)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated or freed by the call"
        for (ctx, top_k, kmax), buf, ref in zip(problems, outs, refs):
            assert torch.equal(buf.sel_idx, ref.sel_idx), f"rep {rep}: mask differs"
            assert torch.equal(buf.sel_cnt, ref.sel_cnt)
            assert torch.equal(buf.scores.view(torch.int32), ref.scores.view(torch.int32)), f"rep {rep}: scores differ"
    assert li.launch_count() > launches_before             # the library's own kernels ran
    # the mask drives li_sparse_attn exactly as the workspace path's does
    for (ctx, top_k, kmax), buf, ref in zip(problems, outs, refs):
        li.li_sparse_attn(ctx, buf.sel_idx, buf.sel_cnt, kmax, buf.o, buf.lse, buf.workspace)
        torch.cuda.synchronize()
        assert torch.equal(buf.o.view(torch.int16), ref.o.view(torch.int16))
        assert torch.equal(buf.lse.view(torch.int32), ref.lse.view(torch.int32))
