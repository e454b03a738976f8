"""paper_2605_31158_b200 -- thin ctypes binding over libli.so (include/li.h).

Argument marshalling only: every step of the hot path (pooling, scoring, top-k, paged gather, attention)
runs in the CUDA kernels of csrc/.  torch is used for device memory and streams.  There is no CPU fallback:
if libli.so is missing or cannot be loaded, every call raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence, Tuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libli.so")

LI_OK, LI_ERR_INVALID_ARG, LI_ERR_UNSUPPORTED, LI_ERR_WORKSPACE, LI_ERR_CUDA, LI_ERR_TOO_LARGE = 0, -1, -2, -3, -4, -5
LI_STATIC_SCRATCH_BYTES = 16 << 20
LI_MAX_CALLS = 64
LI_FLAG_NO_SPLIT = 1
LI_FLAG_KV_FP8 = 2
LI_BAD_PAGE_ID, LI_BAD_SEL_CNT, LI_BAD_SEL_RANGE, LI_BAD_SEL_DUPLICATE = 1, 2, 4, 8

EXPORTS = ("li_block_select", "li_block_select_reuse_kbar", "li_block_select_cached", "li_block_select_static",
           "li_static_scratch_needed", "li_pool_pages", "li_slice_cache_bytes",
           "li_sparse_attn", "li_validate", "li_quantize_pages", "li_workspace_bytes", "li_context_policy",
           "li_policy_workspace_bytes", "li_launch_count", "li_reset_launch_count", "li_strerror", "li_version",
           "li_last_cuda_error")


class LiError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        extra = f", cudaError {lib().li_last_cuda_error()}" if code == LI_ERR_CUDA else ""
        super().__init__(f"{where}: {strerror(code)} ({code}{extra})")


class li_problem(ctypes.Structure):
    """Mirror of `struct li_problem` in include/li.h."""
    _fields_ = [
        ("B", ctypes.c_int32), ("H", ctypes.c_int32), ("Lq", ctypes.c_int32), ("d", ctypes.c_int32),
        ("frame_tokens", ctypes.c_int32), ("block_q", ctypes.c_int32), ("block_k", ctypes.c_int32),
        ("n_pages", ctypes.c_int32),
        ("q", ctypes.c_void_p), ("q_sb", ctypes.c_int64), ("q_sh", ctypes.c_int64), ("q_st", ctypes.c_int64),
        ("k_cache", ctypes.c_void_p), ("v_cache", ctypes.c_void_p),
        ("kv_sp", ctypes.c_int64), ("kv_sh", ctypes.c_int64), ("kv_st", ctypes.c_int64),
        ("frame_idx", ctypes.c_void_p), ("frame_off_host", ctypes.c_void_p),
        ("n_cur_frames", ctypes.c_int32), ("softmax_scale", ctypes.c_float),
        ("grid_h", ctypes.c_int32), ("grid_w", ctypes.c_int32),
        ("bt", ctypes.c_int32), ("bh", ctypes.c_int32), ("bw", ctypes.c_int32),
        ("Lt", ctypes.c_int32), ("text_k", ctypes.c_void_p), ("text_v", ctypes.c_void_p),
        ("t_sb", ctypes.c_int64), ("t_sh", ctypes.c_int64), ("t_st", ctypes.c_int64),
        ("flags", ctypes.c_uint32),
        ("k_scale", ctypes.c_void_p), ("v_scale", ctypes.c_void_p),
    ]


class li_policy(ctypes.Structure):
    """Mirror of `struct li_policy` in include/li.h."""
    _fields_ = [
        ("z_prev1", ctypes.c_void_p), ("z_prev2", ctypes.c_void_p), ("n_latent", ctypes.c_int64),
        ("latent_bf16", ctypes.c_int32), ("alpha", ctypes.c_float), ("kappa", ctypes.c_float),
        ("L_max", ctypes.c_int32), ("round_nearest", ctypes.c_int32), ("ema_state", ctypes.c_void_p),
        ("s_pose", ctypes.c_void_p), ("n_cand", ctypes.c_int32), ("tau_pose", ctypes.c_float),
        ("mem_pages", ctypes.c_void_p), ("n_mem", ctypes.c_int32),
        ("win_pages", ctypes.c_void_p), ("n_win", ctypes.c_int32),
        ("cur_pages", ctypes.c_void_p), ("n_cur", ctypes.c_int32),
    ]


class li_policy_result(ctypes.Structure):
    """Mirror of `struct li_policy_result` in include/li.h (24 bytes, written to device memory)."""
    _fields_ = [("D_t", ctypes.c_float), ("D_bar", ctypes.c_float), ("L_t", ctypes.c_int32),
                ("keep_memory", ctypes.c_int32), ("n_hist_frames", ctypes.c_int32), ("n_frames", ctypes.c_int32)]


_lib = None


def lib() -> ctypes.CDLL:
    """Loads libli.so (never builds, never falls back)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2605_31158_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        P = ctypes.POINTER(li_problem)
        L.li_workspace_bytes.restype = ctypes.c_size_t
        L.li_workspace_bytes.argtypes = [P, ctypes.c_int32]
        L.li_block_select.restype = ctypes.c_int
        L.li_block_select.argtypes = [P, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p,
                                      ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_size_t,
                                      ctypes.c_void_p]
        L.li_block_select_reuse_kbar.restype = ctypes.c_int
        L.li_block_select_reuse_kbar.argtypes = L.li_block_select.argtypes
        L.li_block_select_static.restype = ctypes.c_int
        L.li_block_select_static.argtypes = [P, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p,
                                             ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p]
        L.li_static_scratch_needed.restype = ctypes.c_size_t
        L.li_static_scratch_needed.argtypes = [P]
        L.li_sparse_attn.restype = ctypes.c_int
        L.li_sparse_attn.argtypes = [P, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p,
                                     ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
        L.li_slice_cache_bytes.restype = ctypes.c_size_t
        L.li_slice_cache_bytes.argtypes = [P]
        L.li_pool_pages.restype = ctypes.c_int
        L.li_pool_pages.argtypes = [P, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p]
        L.li_block_select_cached.restype = ctypes.c_int
        L.li_block_select_cached.argtypes = [P, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p,
                                             ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p,
                                             ctypes.c_size_t, ctypes.c_void_p]
        L.li_policy_workspace_bytes.restype = ctypes.c_size_t
        L.li_policy_workspace_bytes.argtypes = []
        L.li_context_policy.restype = ctypes.c_int
        L.li_context_policy.argtypes = [ctypes.POINTER(li_policy), ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p,
                                        ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
        L.li_quantize_pages.restype = ctypes.c_int
        L.li_quantize_pages.argtypes = [P, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p]
        L.li_validate.restype = ctypes.c_int
        L.li_validate.argtypes = [P, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p]
        L.li_last_cuda_error.restype = ctypes.c_int
        L.li_last_cuda_error.argtypes = []
        L.li_launch_count.restype = ctypes.c_int64
        L.li_reset_launch_count.restype = None
        L.li_strerror.restype = ctypes.c_char_p
        L.li_strerror.argtypes = [ctypes.c_int]
        L.li_version.restype = ctypes.c_int
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().li_strerror(int(code)).decode()


def version() -> int:
    return int(lib().li_version())


def launch_count() -> int:
    return int(lib().li_launch_count())


def reset_launch_count() -> None:
    lib().li_reset_launch_count()


class Context:
    """Holds one li_problem plus the host arrays it points to (kept alive for the lifetime of the object)."""

    def __init__(self, q: torch.Tensor, k_cache: torch.Tensor, v_cache: torch.Tensor, frame_idx: torch.Tensor,
                 frame_off: Sequence[int], n_cur_frames: int, block: int, softmax_scale: float = 0.0,
                 grid: Optional[Tuple[int, int]] = None, block3d: Optional[Tuple[int, int, int]] = None,
                 text_k: Optional[torch.Tensor] = None, text_v: Optional[torch.Tensor] = None, flags: int = 0,
                 k_scale: Optional[torch.Tensor] = None, v_scale: Optional[torch.Tensor] = None):
        """k_cache / v_cache: bf16, or uint8 FP8-E4M3 codes together with k_scale / v_scale (fp32 CUDA tensors [H])."""
        fp8 = k_cache.dtype == torch.uint8
        for t, name, dt in ((q, "q", torch.bfloat16), (k_cache, "k_cache", torch.uint8 if fp8 else torch.bfloat16),
                            (v_cache, "v_cache", torch.uint8 if fp8 else torch.bfloat16)):
            if t.dtype != dt or not t.is_cuda or t.dim() != 4 or t.stride(-1) != 1:
                raise ValueError(f"{name} must be a 4-D CUDA {dt} tensor with unit innermost stride")
        if fp8:
            for t, name in ((k_scale, "k_scale"), (v_scale, "v_scale")):
                if t is None or t.dtype != torch.float32 or not t.is_cuda or not t.is_contiguous() or t.numel() != q.shape[1]:
                    raise ValueError(f"{name} must be a contiguous fp32 CUDA tensor of H entries")
            flags |= LI_FLAG_KV_FP8
        self.k_scale, self.v_scale = k_scale, v_scale
        if k_cache.shape != v_cache.shape or k_cache.stride() != v_cache.stride():
            raise ValueError("k_cache and v_cache must have the same shape and strides")
        if frame_idx.dtype != torch.int32 or not frame_idx.is_cuda or not frame_idx.is_contiguous():
            raise ValueError("frame_idx must be a contiguous CUDA int32 tensor")
        self.q, self.k_cache, self.v_cache, self.frame_idx = q, k_cache, v_cache, frame_idx
        self.frame_off = np.ascontiguousarray(np.asarray(frame_off, dtype=np.int32))
        B, H, Lq, d = q.shape
        if len(self.frame_off) != B + 1:
            raise ValueError("frame_off must have B+1 entries")
        p = li_problem()
        p.B, p.H, p.Lq, p.d = B, H, Lq, d
        p.frame_tokens = k_cache.shape[2]
        p.block_q = p.block_k = block
        p.n_pages = k_cache.shape[0]
        p.q = q.data_ptr()
        p.q_sb, p.q_sh, p.q_st = q.stride(0), q.stride(1), q.stride(2)
        p.k_cache, p.v_cache = k_cache.data_ptr(), v_cache.data_ptr()
        p.kv_sp, p.kv_sh, p.kv_st = k_cache.stride(0), k_cache.stride(1), k_cache.stride(2)
        p.frame_idx = frame_idx.data_ptr()
        p.frame_off_host = self.frame_off.ctypes.data
        p.n_cur_frames = n_cur_frames
        p.softmax_scale = softmax_scale
        p.flags = int(flags)
        if fp8:
            p.k_scale, p.v_scale = k_scale.data_ptr(), v_scale.data_ptr()
        self.text_k, self.text_v = text_k, text_v
        if text_k is not None:
            for t, name in ((text_k, "text_k"), (text_v, "text_v")):
                if t.dtype != torch.bfloat16 or not t.is_cuda or t.dim() != 4 or t.stride(-1) != 1:
                    raise ValueError(f"{name} must be a 4-D CUDA bf16 tensor with unit innermost stride")
            if text_k.shape != text_v.shape or text_k.stride() != text_v.stride() or text_k.shape[:2] != (B, H):
                raise ValueError("text_k / text_v must both be [B,H,Lt,d] with equal strides")
            p.Lt = text_k.shape[2]
            p.text_k, p.text_v = text_k.data_ptr(), text_v.data_ptr()
            p.t_sb, p.t_sh, p.t_st = text_k.stride(0), text_k.stride(1), text_k.stride(2)
        self.p = p
        self.B, self.H, self.Lq, self.d, self.block = B, H, Lq, d, block
        n_hist = (self.frame_off[1:] - self.frame_off[:-1]) - n_cur_frames
        if block3d is not None:
            (p.grid_h, p.grid_w), (p.bt, p.bh, p.bw) = grid, block3d
            per_group = (-(-p.grid_h // p.bh)) * (-(-p.grid_w // p.bw))
            self.Nqb = -(-(Lq // p.frame_tokens) // p.bt) * per_group
            self.M = [-(-int(n) // p.bt) * per_group for n in n_hist]
        else:
            self.Nqb = -(-Lq // block)
            self.M = [-(-(int(n) * p.frame_tokens) // block) for n in n_hist]
        self.Mmax = max(self.M) if self.M else 0

    def workspace_bytes(self, kmax: int) -> int:
        n = int(lib().li_workspace_bytes(ctypes.byref(self.p), int(kmax)))
        if n == 0:
            raise LiError(LI_ERR_INVALID_ARG, "li_workspace_bytes")
        return n


def _stream_ptr(stream: Optional[torch.cuda.Stream]) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def li_workspace_bytes(ctx: Context, kmax: int) -> int:
    return ctx.workspace_bytes(kmax)


def li_block_select(ctx: Context, top_k: Sequence[int], kmax: int, sel_idx: torch.Tensor, sel_cnt: torch.Tensor,
                    workspace: torch.Tensor, scores: Optional[torch.Tensor] = None,
                    stream: Optional[torch.cuda.Stream] = None, reuse_kbar: bool = False) -> None:
    """li_block_select / li_block_select_reuse_kbar (include/li.h).  sel_idx int32 [B,H,Nqb,kmax], sel_cnt int32 [B,H,Nqb],
    scores None or fp32 [B,H,Nqb,pitch]; workspace: uint8 CUDA tensor of >= li_workspace_bytes."""
    tk = np.ascontiguousarray(np.asarray(top_k, dtype=np.int32))
    if len(tk) != ctx.B:
        raise ValueError("top_k must have B entries")
    pitch = int(scores.shape[-1]) if scores is not None else 0
    fn = lib().li_block_select_reuse_kbar if reuse_kbar else lib().li_block_select
    rc = fn(ctypes.byref(ctx.p), tk.ctypes.data, int(kmax), sel_idx.data_ptr(),
                               sel_cnt.data_ptr(), scores.data_ptr() if scores is not None else None, pitch,
                               workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                               _stream_ptr(stream))
    if rc != LI_OK:
        raise LiError(rc, "li_block_select")


def li_block_select_static(ctx: Context, top_k: Sequence[int], kmax: int, sel_idx: torch.Tensor, sel_cnt: torch.Tensor,
                           scores: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None) -> None:
    """li_block_select_static (include/li.h): li_block_select without a workspace argument and without any allocation; the
    scratch is a LI_STATIC_SCRATCH_BYTES array inside libli.so shared by all calls (LiError LI_ERR_TOO_LARGE beyond it)."""
    tk = np.ascontiguousarray(np.asarray(top_k, dtype=np.int32))
    if len(tk) != ctx.B:
        raise ValueError("top_k must have B entries")
    pitch = int(scores.shape[-1]) if scores is not None else 0
    rc = lib().li_block_select_static(ctypes.byref(ctx.p), tk.ctypes.data, int(kmax), sel_idx.data_ptr(), sel_cnt.data_ptr(),
                                      scores.data_ptr() if scores is not None else None, pitch, _stream_ptr(stream))
    if rc != LI_OK:
        raise LiError(rc, "li_block_select_static")


def li_static_scratch_needed(ctx: Context) -> int:
    return int(lib().li_static_scratch_needed(ctypes.byref(ctx.p)))


def li_slice_cache_bytes(ctx: Context) -> int:
    return int(lib().li_slice_cache_bytes(ctypes.byref(ctx.p)))


def li_pool_pages(ctx: Context, pages: torch.Tensor, slice_cache: torch.Tensor,
                  stream: Optional[torch.cuda.Stream] = None) -> None:
    """li_pool_pages (include/li.h): patch sums of the listed K pages (int32 CUDA tensor) into slice_cache (fp32 CUDA
    tensor of li_slice_cache_bytes bytes).  3-D tiling only."""
    if pages.dtype != torch.int32 or not pages.is_cuda or not pages.is_contiguous():
        raise ValueError("pages must be a contiguous int32 CUDA tensor")
    if slice_cache.dtype != torch.float32 or not slice_cache.is_cuda or not slice_cache.is_contiguous() or \
            slice_cache.numel() * 4 < li_slice_cache_bytes(ctx):
        raise ValueError("slice_cache must be a contiguous fp32 CUDA tensor of li_slice_cache_bytes bytes")
    rc = lib().li_pool_pages(ctypes.byref(ctx.p), pages.data_ptr(), pages.numel(), slice_cache.data_ptr(), _stream_ptr(stream))
    if rc != LI_OK:
        raise LiError(rc, "li_pool_pages")


def li_block_select_cached(ctx: Context, top_k: Sequence[int], kmax: int, sel_idx: torch.Tensor, sel_cnt: torch.Tensor,
                           slice_cache: torch.Tensor, workspace: torch.Tensor, scores: Optional[torch.Tensor] = None,
                           stream: Optional[torch.cuda.Stream] = None) -> None:
    """li_block_select_cached (include/li.h): li_block_select with the historical block means formed from slice_cache."""
    tk = np.ascontiguousarray(np.asarray(top_k, dtype=np.int32))
    if len(tk) != ctx.B:
        raise ValueError("top_k must have B entries")
    pitch = int(scores.shape[-1]) if scores is not None else 0
    rc = lib().li_block_select_cached(ctypes.byref(ctx.p), tk.ctypes.data, int(kmax), sel_idx.data_ptr(), sel_cnt.data_ptr(),
                                      scores.data_ptr() if scores is not None else None, pitch, slice_cache.data_ptr(),
                                      workspace.data_ptr(), workspace.numel() * workspace.element_size(), _stream_ptr(stream))
    if rc != LI_OK:
        raise LiError(rc, "li_block_select_cached")


def li_sparse_attn(ctx: Context, sel_idx: torch.Tensor, sel_cnt: torch.Tensor, kmax: int, o: torch.Tensor,
                   lse: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
                   stream: Optional[torch.cuda.Stream] = None) -> None:
    """li_sparse_attn (include/li.h).  o bf16 [B,H,Lq,d] contiguous; lse None or fp32 [B,H,Lq]."""
    rc = lib().li_sparse_attn(ctypes.byref(ctx.p), sel_idx.data_ptr(), sel_cnt.data_ptr(), int(kmax), o.data_ptr(),
                              lse.data_ptr() if lse is not None else None,
                              workspace.data_ptr() if workspace is not None else None,
                              workspace.numel() * workspace.element_size() if workspace is not None else 0,
                              _stream_ptr(stream))
    if rc != LI_OK:
        raise LiError(rc, "li_sparse_attn")


def li_quantize_pages(ctx: Context, k_src: torch.Tensor, v_src: torch.Tensor, pages: torch.Tensor,
                      stream: Optional[torch.cuda.Stream] = None) -> None:
    """li_quantize_pages (include/li.h): bf16 rows [n_list,H,T_f,d] -> the FP8 pages `pages` (int32 CUDA) of ctx's caches."""
    for t in (k_src, v_src):
        if t.dtype != torch.bfloat16 or not t.is_cuda or not t.is_contiguous() or t.shape[1:] != ctx.k_cache.shape[1:] or \
                t.shape[0] != pages.numel():
            raise ValueError("k_src / v_src must be contiguous bf16 CUDA tensors [n_list,H,T_f,d]")
    if pages.dtype != torch.int32 or not pages.is_cuda or not pages.is_contiguous():
        raise ValueError("pages must be a contiguous int32 CUDA tensor")
    rc = lib().li_quantize_pages(ctypes.byref(ctx.p), k_src.data_ptr(), v_src.data_ptr(), pages.data_ptr(), pages.numel(),
                                 _stream_ptr(stream))
    if rc != LI_OK:
        raise LiError(rc, "li_quantize_pages")


def li_validate(ctx: Context, error: torch.Tensor, sel_idx: Optional[torch.Tensor] = None,
                sel_cnt: Optional[torch.Tensor] = None, kmax: int = 0, stream: Optional[torch.cuda.Stream] = None) -> None:
    """li_validate (include/li.h): device-side check of the frame lists (and of sel_idx / sel_cnt when given) into
    `error`, an int32 CUDA tensor of 4 entries: [LI_BAD_* bits, 1 + call, position, value]."""
    if error.dtype != torch.int32 or not error.is_cuda or error.numel() < 4 or not error.is_contiguous():
        raise ValueError("error must be a contiguous int32 CUDA tensor of >= 4 entries")
    rc = lib().li_validate(ctypes.byref(ctx.p), sel_idx.data_ptr() if sel_idx is not None else None,
                           sel_cnt.data_ptr() if sel_cnt is not None else None, int(kmax), error.data_ptr(),
                           _stream_ptr(stream))
    if rc != LI_OK:
        raise LiError(rc, "li_validate")


class Buffers:
    """Output/workspace tensors for one Context (allocated once by the caller, reused across calls)."""

    def __init__(self, ctx: Context, kmax: int, want_scores: bool = False, want_lse: bool = True):
        dev = ctx.q.device
        self.kmax = int(kmax)
        self.sel_idx = torch.empty((ctx.B, ctx.H, ctx.Nqb, self.kmax), dtype=torch.int32, device=dev)
        self.sel_cnt = torch.empty((ctx.B, ctx.H, ctx.Nqb), dtype=torch.int32, device=dev)
        self.scores = (torch.empty((ctx.B, ctx.H, ctx.Nqb, max(1, ctx.Mmax)), dtype=torch.float32, device=dev)
                       if want_scores else None)
        self.workspace = torch.empty((ctx.workspace_bytes(self.kmax),), dtype=torch.uint8, device=dev)
        self.o = torch.empty((ctx.B, ctx.H, ctx.Lq, ctx.d), dtype=torch.bfloat16, device=dev)
        self.lse = torch.empty((ctx.B, ctx.H, ctx.Lq), dtype=torch.float32, device=dev) if want_lse else None


def forward(ctx: Context, top_k: Sequence[int], buf: Buffers,
            stream: Optional[torch.cuda.Stream] = None) -> Tuple[torch.Tensor, Optional[torch.Tensor]]:
    """One pass of the whole hot path: li_block_select then li_sparse_attn (two C-ABI calls)."""
    li_block_select(ctx, top_k, buf.kmax, buf.sel_idx, buf.sel_cnt, buf.workspace, buf.scores, stream)
    li_sparse_attn(ctx, buf.sel_idx, buf.sel_cnt, buf.kmax, buf.o, buf.lse, buf.workspace, stream)
    return buf.o, buf.lse


def li_context_policy(z_prev1: torch.Tensor, z_prev2: torch.Tensor, ema_state: torch.Tensor, alpha: float, kappa: float,
                      L_max: int, s_pose: Optional[torch.Tensor], tau_pose: float, mem_pages: Optional[torch.Tensor],
                      win_pages: Optional[torch.Tensor], cur_pages: torch.Tensor, frame_idx_out: torch.Tensor,
                      result: torch.Tensor, workspace: torch.Tensor, round_nearest: bool = False,
                      stream: Optional[torch.cuda.Stream] = None) -> None:
    """li_context_policy (include/li.h; Eq. 1-4).  All tensors live on the GPU: latents fp32 or bf16 (contiguous),
    ema_state fp32 [2], s_pose fp32 [n_cand], page lists int32, frame_idx_out int32 [capacity], result uint8 [24]
    (read it with `policy_result`), workspace uint8 [>= li_policy_workspace_bytes]."""
    if z_prev1.shape != z_prev2.shape or z_prev1.dtype != z_prev2.dtype or z_prev1.dtype not in (torch.float32, torch.bfloat16):
        raise ValueError("latents must be two fp32 or bf16 tensors of the same shape")
    tensors = [z_prev1, z_prev2, ema_state, cur_pages, frame_idx_out, result, workspace] + \
              [t for t in (s_pose, mem_pages, win_pages) if t is not None]
    if not all(t.is_cuda and t.is_contiguous() for t in tensors):
        raise ValueError("li_context_policy takes contiguous CUDA tensors")
    for t, dt, name in ((ema_state, torch.float32, "ema_state"), (s_pose, torch.float32, "s_pose"),
                        (mem_pages, torch.int32, "mem_pages"), (win_pages, torch.int32, "win_pages"),
                        (cur_pages, torch.int32, "cur_pages"), (frame_idx_out, torch.int32, "frame_idx_out")):
        if t is not None and t.dtype != dt:
            raise ValueError(f"{name} must be {dt}")
    if ema_state.numel() < 2 or result.numel() * result.element_size() < ctypes.sizeof(li_policy_result):
        raise ValueError("ema_state needs 2 floats, result 24 bytes")
    pp = li_policy()
    pp.z_prev1, pp.z_prev2, pp.n_latent = z_prev1.data_ptr(), z_prev2.data_ptr(), z_prev1.numel()
    pp.latent_bf16 = 1 if z_prev1.dtype == torch.bfloat16 else 0
    pp.alpha, pp.kappa, pp.L_max, pp.round_nearest = float(alpha), float(kappa), int(L_max), 1 if round_nearest else 0
    pp.ema_state = ema_state.data_ptr()
    pp.s_pose, pp.n_cand, pp.tau_pose = (s_pose.data_ptr() if s_pose is not None else None,
                                         s_pose.numel() if s_pose is not None else 0, float(tau_pose))
    pp.mem_pages, pp.n_mem = (mem_pages.data_ptr(), mem_pages.numel()) if mem_pages is not None else (None, 0)
    pp.win_pages, pp.n_win = (win_pages.data_ptr(), win_pages.numel()) if win_pages is not None else (None, 0)
    pp.cur_pages, pp.n_cur = cur_pages.data_ptr(), cur_pages.numel()
    rc = lib().li_context_policy(ctypes.byref(pp), frame_idx_out.data_ptr(), frame_idx_out.numel(), result.data_ptr(),
                                 workspace.data_ptr(), workspace.numel() * workspace.element_size(), _stream_ptr(stream))
    if rc != LI_OK:
        raise LiError(rc, "li_context_policy")


def policy_result(result: torch.Tensor) -> li_policy_result:
    """Copies the 24-byte li_policy_result record to the host (synchronises on the copy)."""
    raw = result.cpu().numpy().tobytes()[:ctypes.sizeof(li_policy_result)]
    return li_policy_result.from_buffer_copy(raw)
