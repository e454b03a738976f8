"""CPU-only checks of the boundary: libli.so builds for sm_100a, loads, exports every function include/li.h
declares, and rejects bad arguments on the host before any CUDA call (no compute without a GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2605_31158_b200 as li
from paper_2605_31158_b200 import build as libuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    libuild.build()
    return li.lib()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "li.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(li_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    names = declared_functions()
    assert set(names) == set(li.EXPORTS)
    for n in names:
        assert getattr(L, n) is not None
    assert li.version() == 200
    assert li.strerror(0) == "ok" and "unsupported" in li.strerror(li.LI_ERR_UNSUPPORTED)


def test_sass_contains_tcgen05_and_tma():
    """The attention kernel must be the Blackwell-native path: UTC*MMA (tcgen05.mma), LDTM/STTM, UTMALDG (TMA)."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    libuild.build()
    sass = subprocess.run([cuobjdump, "-sass", li.LIB_PATH], capture_output=True, text=True).stdout
    for mnemonic in ("UTCHMMA", "LDTM", "STTM", "UTMALDG"):
        assert mnemonic in sass, mnemonic
    assert "HMMA.16816" not in sass            # no legacy mma.sync path


def make_problem(**over):
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


def test_workspace_bytes_and_validation(L):
    p, fo = make_problem()
    ws = L.li_workspace_bytes(ctypes.byref(p), 8)
    # qbar [1,2,4,64] fp32 + kbar [1,2,64,32] fp32 (transposed, M padded to 32) + score keys [1,2,4,12] u32,
    # each rounded up to 256 B
    # + the attention kernel's split buffers: 320 slots x 128 rows x (d fp32 + one float2)
    assert ws == 2 * 4 * 64 * 4 + 2 * 64 * 32 * 4 + 512 + 320 * 128 * (64 * 4 + 8)
    tk = np.asarray([8], dtype=np.int32)

    def select(prob, kmax=8, ws_ptr=0x50000, ws_bytes=ws, sel=0x60000, cnt=0x70000):
        return L.li_block_select(ctypes.byref(prob), tk.ctypes.data, kmax, sel, cnt, None, 0, ws_ptr, ws_bytes, None)

    def attn(prob, o=0x80000):
        return L.li_sparse_attn(ctypes.byref(prob), 0x60000, 0x70000, 8, o, None, None, 0, None)

    for bad, code in ((dict(d=96), li.LI_ERR_UNSUPPORTED), (dict(block_q=128), li.LI_ERR_UNSUPPORTED),
                      (dict(block_q=32, block_k=32), li.LI_ERR_UNSUPPORTED), (dict(B=65), li.LI_ERR_UNSUPPORTED),
                      (dict(frame_tokens=250), li.LI_ERR_INVALID_ARG), (dict(q=0), li.LI_ERR_INVALID_ARG),
                      (dict(q=0x10008), li.LI_ERR_INVALID_ARG), (dict(kv_st=60), li.LI_ERR_INVALID_ARG),
                      (dict(Lq=100), li.LI_ERR_INVALID_ARG), (dict(n_cur_frames=5), li.LI_ERR_INVALID_ARG),
                      (dict(softmax_scale=-1.0), li.LI_ERR_INVALID_ARG), (dict(H=0), li.LI_ERR_INVALID_ARG)):
        pb, keep = make_problem(**bad)
        assert select(pb) == code, bad
        assert attn(pb) == code, bad
        assert L.li_workspace_bytes(ctypes.byref(pb), 8) == 0
    assert select(p, kmax=4) == li.LI_ERR_INVALID_ARG           # kmax < k_b
    assert select(p, ws_bytes=ws - 1) == li.LI_ERR_WORKSPACE
    assert select(p, ws_ptr=0) == li.LI_ERR_WORKSPACE
    assert select(p, ws_ptr=0x50010) == li.LI_ERR_WORKSPACE     # not 256-byte aligned
    assert select(p, sel=0) == li.LI_ERR_INVALID_ARG
    assert attn(p, o=0) == li.LI_ERR_INVALID_ARG
    assert L.li_block_select(None, tk.ctypes.data, 8, 1, 1, None, 0, 1, 1, None) == li.LI_ERR_INVALID_ARG


def test_3d_tiling_validation(L):
    """3-D block fields: accepted geometries and host-side rejections."""
    def prob3d(**over):
        fo = np.asarray([0, 6], dtype=np.int32)
        p, _ = make_problem(frame_tokens=30 * 52, Lq=2 * 30 * 52, d=128, block_q=128, block_k=128, n_cur_frames=2,
                            q_sb=24 * 3120 * 128, q_sh=3120 * 128, q_st=128, kv_sp=24 * 1560 * 128, kv_sh=1560 * 128,
                            kv_st=128, H=24, grid_h=30, grid_w=52, bt=4, bh=8, bw=4)
        p.frame_off_host = fo.ctypes.data
        for k, v in over.items():
            setattr(p, k, v)
        return p, fo
    p, keep = prob3d()
    # history 4 frames -> 1 temporal group x 4 x 13 = 52 blocks; Nqb = 52 (chunk of 2 frames = one partial group)
    ws = L.li_workspace_bytes(ctypes.byref(p), 8)
    assert ws == (24 * 52 * 128 * 4 + 24 * 128 * 64 * 4 + 24 * 52 * 52 * 4 + (256 - (24 * 52 * 52 * 4) % 256) % 256
                  + 320 * 128 * (128 * 4 + 8))
    for bad, code in ((dict(bw=8), li.LI_ERR_UNSUPPORTED),            # 4*8*8 != 128
                      (dict(bh=4, bw=8), li.LI_OK),                    # (4,4,8) on a 52-wide grid: partial right border
                      (dict(bh=16, bw=2), li.LI_OK),                   # any bh*bw == 32
                      (dict(bh=8, bw=8, bt=2), li.LI_ERR_UNSUPPORTED), # bh*bw != 32
                      (dict(grid_w=50), li.LI_ERR_INVALID_ARG),        # grid_h*grid_w != frame_tokens
                      (dict(bt=0), li.LI_ERR_INVALID_ARG),             # partially specified
                      (dict(bt=2, block_q=64, block_k=64), li.LI_OK)): # (2,8,4) = 64-token blocks
        pb, keep2 = prob3d(**bad)
        got = L.li_workspace_bytes(ctypes.byref(pb), 8)
        assert (got > 0) == (code == li.LI_OK), bad
        if code != li.LI_OK:
            assert L.li_sparse_attn(ctypes.byref(pb), 0x60000, 0x70000, 8, 0x80000, None, None, 0, None) == code, bad


def test_text_prefix_validation(L):
    p, fo = make_problem(Lt=77, text_k=0x90000, text_v=0xA0000, t_sb=2 * 77 * 64, t_sh=77 * 64, t_st=64)
    assert L.li_workspace_bytes(ctypes.byref(p), 8) > 0
    for bad in (dict(text_k=0), dict(text_v=0x90008), dict(t_st=60), dict(t_sh=0), dict(Lt=-1)):
        pb, keep = make_problem(**{**dict(Lt=77, text_k=0x90000, text_v=0xA0000, t_sb=2 * 77 * 64, t_sh=77 * 64, t_st=64), **bad})
        assert L.li_workspace_bytes(ctypes.byref(pb), 8) == 0, bad
        assert L.li_sparse_attn(ctypes.byref(pb), 0x60000, 0x70000, 8, 0x80000, None, None, 0, None) == li.LI_ERR_INVALID_ARG, bad


def test_binding_refuses_cpu_tensors():
    import torch
    q = torch.zeros((1, 2, 256, 64), dtype=torch.bfloat16)
    kc = torch.zeros((8, 2, 256, 64), dtype=torch.bfloat16)
    with pytest.raises(ValueError):
        li.Context(q, kc, kc, torch.zeros(4, dtype=torch.int32), [0, 4], 1, 64)


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    monkeypatch.setattr(li, "_lib", None)
    monkeypatch.setattr(li, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        li.lib()


def test_context_policy_validation(L):
    """li_context_policy (Eq. 1-4): host-side argument checks, no launch (pointers are fake device addresses)."""
    def pol(**over):
        pp = li.li_policy()
        pp.z_prev1, pp.z_prev2, pp.n_latent, pp.latent_bf16 = 0x10000, 0x20000, 1000, 0
        pp.alpha, pp.kappa, pp.L_max, pp.round_nearest = 0.5, 0.02, 8, 0
        pp.ema_state = 0x30000
        pp.s_pose, pp.n_cand, pp.tau_pose = 0x40000, 3, 0.45
        pp.mem_pages, pp.n_mem, pp.win_pages, pp.n_win, pp.cur_pages, pp.n_cur = 0x50000, 2, 0x60000, 20, 0x70000, 4
        for k, v in over.items():
            setattr(pp, k, v)
        return pp

    def call(pp, out=0x80000, cap=14, res=0x90000, ws=0xA0000, ws_bytes=None):
        n = L.li_policy_workspace_bytes() if ws_bytes is None else ws_bytes
        return L.li_context_policy(ctypes.byref(pp), out, cap, res, ws, n, None)

    assert L.li_policy_workspace_bytes() == 8192
    for bad in (dict(z_prev1=0), dict(z_prev2=0x20004), dict(n_latent=0), dict(latent_bf16=2), dict(alpha=0.0),
                dict(alpha=1.5), dict(kappa=0.0), dict(L_max=0), dict(ema_state=0), dict(s_pose=0), dict(n_cand=-1),
                dict(mem_pages=0), dict(win_pages=0), dict(cur_pages=0)):
        assert call(pol(**bad)) == li.LI_ERR_INVALID_ARG, bad
    assert call(pol(), cap=13) == li.LI_ERR_INVALID_ARG          # capacity < n_mem + min(L_max, n_win) + n_cur
    assert call(pol(), out=0) == li.LI_ERR_INVALID_ARG
    assert call(pol(), res=0) == li.LI_ERR_INVALID_ARG
    assert call(pol(), ws=0) == li.LI_ERR_WORKSPACE
    assert call(pol(), ws_bytes=100) == li.LI_ERR_WORKSPACE
    assert call(pol(), ws=0xA0010) == li.LI_ERR_WORKSPACE


def test_slice_cache_validation(L):
    """li_pool_pages / li_block_select_cached exist for the 3-D tiling only; host-side argument checks."""
    p1, keep1 = make_problem()                       # 1-D blocks
    assert L.li_slice_cache_bytes(ctypes.byref(p1)) == 0
    assert L.li_pool_pages(ctypes.byref(p1), 0x50000, 1, 0x60000, None) == li.LI_ERR_UNSUPPORTED
    tk = np.asarray([8], dtype=np.int32)
    ws = L.li_workspace_bytes(ctypes.byref(p1), 8)
    assert L.li_block_select_cached(ctypes.byref(p1), tk.ctypes.data, 8, 0x60000, 0x70000, None, 0, 0x90000, 0x50000, ws,
                                    None) == li.LI_ERR_UNSUPPORTED
    fo = np.asarray([0, 6], dtype=np.int32)
    p3, keep3 = make_problem(frame_tokens=30 * 52, Lq=2 * 30 * 52, d=128, block_q=128, block_k=128, n_cur_frames=2,
                             q_sb=24 * 3120 * 128, q_sh=3120 * 128, q_st=128, kv_sp=24 * 1560 * 128, kv_sh=1560 * 128,
                             kv_st=128, H=24, grid_h=30, grid_w=52, bt=4, bh=8, bw=4)
    p3.frame_off_host = fo.ctypes.data
    assert L.li_slice_cache_bytes(ctypes.byref(p3)) == p3.n_pages * 24 * 4 * 13 * 128 * 4
    assert L.li_pool_pages(ctypes.byref(p3), 0, 1, 0x60000, None) == li.LI_ERR_INVALID_ARG
    assert L.li_pool_pages(ctypes.byref(p3), 0x50000, 1, 0, None) == li.LI_ERR_INVALID_ARG
    assert L.li_pool_pages(ctypes.byref(p3), 0x50000, -1, 0x60000, None) == li.LI_ERR_INVALID_ARG
    ws3 = L.li_workspace_bytes(ctypes.byref(p3), 8)
    assert L.li_block_select_cached(ctypes.byref(p3), tk.ctypes.data, 8, 0x60000, 0x70000, None, 0, 0, 0x50000, ws3,
                                    None) == li.LI_ERR_INVALID_ARG


def test_validate_and_flags_argument_checks(L):
    """li_validate (debug check of device-side inputs) and li_problem.flags: host-side rejections."""
    p, fo = make_problem()
    assert L.li_validate(ctypes.byref(p), None, None, 0, None, None) == li.LI_ERR_INVALID_ARG          # no error word
    assert L.li_validate(ctypes.byref(p), 0x60000, None, 8, 0x90000, None) == li.LI_ERR_INVALID_ARG    # sel_idx without sel_cnt
    assert L.li_validate(ctypes.byref(p), None, 0x70000, 8, 0x90000, None) == li.LI_ERR_INVALID_ARG
    assert L.li_validate(ctypes.byref(p), 0x60000, 0x70000, 0, 0x90000, None) == li.LI_ERR_INVALID_ARG  # kmax < 1
    bad, keep = make_problem(d=96)
    assert L.li_validate(ctypes.byref(bad), None, None, 0, 0x90000, None) == li.LI_ERR_UNSUPPORTED
    assert li.LI_FLAG_NO_SPLIT == 1 and li.li_problem.flags.size == 4
    # the struct mirrors include/li.h field for field (flags is the last member)
    hdr = open(os.path.join(ROOT, "include", "li.h")).read()
    body = hdr[hdr.index("typedef struct li_problem {"):hdr.index("} li_problem;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct li_problem {", "").strip()
        if decl:
            names += [n.strip().lstrip("*").strip() for n in re.sub(r"^(const\s+)?\w+(\s+\*?|\s*\*\s*)", "", decl, count=1).split(",")]
    assert names == [f[0] for f in li.li_problem._fields_]


def test_page_pool_entry_points_need_only_the_cache(L):
    """li_slice_cache_bytes / li_pool_pages look at the K cache and the tiling only: Q, the frame lists and their host
    offsets may be absent."""
    p3, keep3 = make_problem(frame_tokens=30 * 52, Lq=0, d=128, block_q=128, block_k=128, n_cur_frames=0, q=0, frame_idx=0,
                             frame_off_host=0, q_sb=0, q_sh=0, q_st=0, kv_sp=24 * 1560 * 128, kv_sh=1560 * 128,
                             kv_st=128, H=24, grid_h=30, grid_w=52, bt=4, bh=8, bw=4)
    assert L.li_slice_cache_bytes(ctypes.byref(p3)) == p3.n_pages * 24 * 4 * 13 * 128 * 4
    assert L.li_pool_pages(ctypes.byref(p3), 0x50000, 0, 0x60000, None) == li.LI_OK                   # empty list: nothing to do
    assert L.li_pool_pages(ctypes.byref(p3), 0x50000, 1, 0x60008, None) == li.LI_ERR_INVALID_ARG      # cache misaligned
    p3.k_cache = 0
    assert L.li_slice_cache_bytes(ctypes.byref(p3)) == 0


def test_no_device_means_cuda_error_not_a_fallback(L):
    """Without a CUDA device a compute call fails with LI_ERR_CUDA and li_last_cuda_error() names the runtime's code:
    there is no CPU path to fall back to.  (Skipped where a GPU is present: the pointers are fake.)"""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    p, fo = make_problem()
    tk = np.asarray([8], dtype=np.int32)
    ws = L.li_workspace_bytes(ctypes.byref(p), 8)
    assert L.li_block_select(ctypes.byref(p), tk.ctypes.data, 8, 0x60000, 0x70000, None, 0, 0x50000, ws, None) == li.LI_ERR_CUDA
    assert L.li_last_cuda_error() != 0


def test_fp8_pages_argument_checks(L):
    """LI_FLAG_KV_FP8 (include/li.h): d = 128 and 128-token blocks only, scales required, byte strides multiples of 16, no text
    prefix, no page-resident patch sums; li_quantize_pages host-side rejections."""
    fo = np.asarray([0, 6], dtype=np.int32)

    def prob8(**over):
        p, _ = make_problem(frame_tokens=1560, Lq=2 * 1560, d=128, block_q=128, block_k=128, n_cur_frames=2, H=24,
                            q_sb=24 * 3120 * 128, q_sh=3120 * 128, q_st=128, kv_sp=24 * 1560 * 128, kv_sh=1560 * 128, kv_st=128,
                            flags=li.LI_FLAG_KV_FP8, k_scale=0xB0000, v_scale=0xC0000)
        p.frame_off_host = fo.ctypes.data
        for k, v in over.items():
            setattr(p, k, v)
        return p

    assert L.li_workspace_bytes(ctypes.byref(prob8()), 8) > 0
    for bad in (dict(d=64, q_st=64, kv_st=64), dict(block_q=64, block_k=64), dict(k_scale=0), dict(v_scale=0), dict(kv_st=136),
                dict(Lt=16, text_k=0x90000, text_v=0xA0000, t_sb=24 * 16 * 128, t_sh=16 * 128, t_st=128)):
        assert L.li_workspace_bytes(ctypes.byref(prob8(**bad)), 8) == 0, bad
    p3 = prob8(grid_h=30, grid_w=52, bt=4, bh=8, bw=4)
    assert L.li_workspace_bytes(ctypes.byref(p3), 8) > 0                   # 3-D blocks are supported with FP8 pages
    assert L.li_slice_cache_bytes(ctypes.byref(p3)) == 0                   # ... page-resident patch sums are not
    assert L.li_pool_pages(ctypes.byref(p3), 0x50000, 1, 0x60000, None) == li.LI_ERR_UNSUPPORTED
    p = prob8()
    q = lambda prob, ks=0x100000, vs=0x200000, pages=0x50000, n=2: L.li_quantize_pages(ctypes.byref(prob), ks, vs, pages, n, None)
    assert q(p, n=0) == li.LI_OK                                           # nothing to do
    assert q(p, ks=0) == li.LI_ERR_INVALID_ARG and q(p, pages=0) == li.LI_ERR_INVALID_ARG and q(p, n=-1) == li.LI_ERR_INVALID_ARG
    assert q(p, vs=0x200008) == li.LI_ERR_INVALID_ARG                      # 16-byte alignment
    assert q(prob8(flags=0)) == li.LI_ERR_INVALID_ARG                      # the problem does not describe FP8 pages
    assert q(prob8(d=64, q_st=64, kv_st=64)) == li.LI_ERR_UNSUPPORTED
