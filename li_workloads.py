"""Seeded synthetic inputs for the Light Interaction sparse-attention hot path.

This module is the ONLY code shared by the CPU oracle's callers and the CUDA path's
callers (tests, bench.py, __graft_entry__.smoke).  It holds none of the method's
arithmetic: it only draws N(0,1) tensors from a seeded torch CPU generator, rounds them
to bf16, lays them out as a frame-paged K/V pool and writes the frame-index list
(retrieved memory | temporal window | current chunk) that PAPER.md:60 (Fig. 2a,
"reconstruct the KV cache for the current chunk") and BASELINE.json's configs describe.

The shapes stand in for the paper's HY-WorldPlay attention workload (480P latent grid
30x52 = 1560 tokens per frame, 4-frame chunks, H=24, d=128, 128-token blocks PAPER.md:321,
retained ratio r PAPER.md:136-138); no VBench item, prompt or checkpoint is used.

Every tensor is generated on the CPU so the very same bits feed the oracle (as uint16
bf16 patterns) and are uploaded for the CUDA path.
"""
from __future__ import annotations

import dataclasses
from fractions import Fraction
from typing import List, Optional, Sequence

import numpy as np
import torch


@dataclasses.dataclass
class Spec:
    """One synthetic workload (a batch of `B = len(n_mem)` independent calls)."""
    name: str
    seed: int
    H: int
    d: int
    frame_tokens: int            # T_f
    n_cur_frames: int            # chunk length in frames; Lq = n_cur_frames * T_f
    block: int                   # block_q == block_k
    n_pages: int                 # pages in the pool
    n_mem: Sequence[int]         # retrieved spatial-memory frames per call
    n_win: Sequence[int]         # temporal-window frames per call
    density: Optional[Fraction] = None   # r of Eq. 10 (history blocks only), exact rational
    top_k: Optional[int] = None          # or a fixed top-k per query-block row
    k_frame_offset_std: float = 0.0      # `long`: per-(page, head) K mean offsets ~ N(0, std^2)
    pages_per_call: Optional[int] = None # adaptive: call b owns pages [b*ppc, (b+1)*ppc)
    explicit_frames: Optional[List[List[int]]] = None  # tiny: frame list given verbatim
    grid: Optional[tuple] = None          # (grid_h, grid_w) of a frame, frame_tokens == grid_h*grid_w   } 3-D blocks,
    block3d: Optional[tuple] = None       # (B_t, B_h, B_w), B_t*B_h*B_w == block                        } PAPER.md:129/:321


@dataclasses.dataclass
class Problem:
    spec: Spec
    q: torch.Tensor              # bf16 [B, H, Lq, d]
    k_cache: torch.Tensor        # bf16 [n_pages, H, T_f, d]
    v_cache: torch.Tensor        # bf16 [n_pages, H, T_f, d]
    frame_idx: np.ndarray        # int32 [sum_b n_frames_b], logical order mem | win | cur
    frame_off: np.ndarray        # int32 [B+1]
    top_k: np.ndarray            # int32 [B]  (already clamped to M_b)

    # ---- derived integers (no floating point) ----
    @property
    def B(self) -> int:
        return len(self.frame_off) - 1

    @property
    def Lq(self) -> int:
        return self.spec.n_cur_frames * self.spec.frame_tokens

    def n_hist_frames(self, b: int) -> int:
        return int(self.frame_off[b + 1] - self.frame_off[b]) - self.spec.n_cur_frames

    def L_hist(self, b: int) -> int:
        return self.n_hist_frames(b) * self.spec.frame_tokens

    def n_blocks(self, n_frames: int) -> int:
        """Blocks of a region of n_frames frames (integer bookkeeping of the tiling)."""
        s = self.spec
        if s.block3d is not None:
            (gh, gw), (bt, bh, bw) = s.grid, s.block3d
            return -(-n_frames // bt) * (-(-gh // bh)) * (-(-gw // bw))
        return -(-(n_frames * s.frame_tokens) // s.block)

    def block_sizes(self, n_frames: int) -> np.ndarray:
        """Valid (non-padding) tokens of every block of a region of n_frames frames."""
        s = self.spec
        if s.block3d is not None:
            (gh, gw), (bt, bh, bw) = s.grid, s.block3d
            ft = [min(bt, n_frames - t * bt) for t in range(-(-n_frames // bt))]
            fh = [min(bh, gh - y * bh) for y in range(-(-gh // bh))]
            fw = [min(bw, gw - x * bw) for x in range(-(-gw // bw))]
            return np.asarray([a * b_ * c for a in ft for b_ in fh for c in fw], dtype=np.int64)
        L = n_frames * s.frame_tokens
        return np.asarray([min(s.block, L - m * s.block) for m in range(-(-L // s.block))], dtype=np.int64)

    def M(self, b: int) -> int:
        return self.n_blocks(self.n_hist_frames(b))

    @property
    def Nqb(self) -> int:
        return self.n_blocks(self.spec.n_cur_frames)

    @property
    def Nc(self) -> int:
        return self.n_blocks(self.spec.n_cur_frames)

    @property
    def kmax(self) -> int:
        return max(1, int(self.top_k.max()) if len(self.top_k) else 1)

    def u16(self, t: torch.Tensor) -> np.ndarray:
        """bf16 tensor -> numpy uint16 bit patterns (what the oracle consumes)."""
        return t.view(torch.int16).numpy().view(np.uint16)


def _randn_bf16(gen: torch.Generator, shape) -> torch.Tensor:
    return torch.randn(shape, generator=gen, dtype=torch.float32).to(torch.bfloat16)


def top_k_for(spec: Spec, M: int) -> int:
    """floor(r*M) in exact rational arithmetic (Eq. 10), or the fixed top-k;
    clamped to M."""
    if spec.top_k is not None:
        k = spec.top_k
    else:
        r = Fraction(spec.density)
        k = (r.numerator * M) // r.denominator
    return min(M, k)


def build(spec: Spec) -> Problem:
    gen = torch.Generator().manual_seed(spec.seed)
    B = len(spec.n_mem)
    T_f, H, d = spec.frame_tokens, spec.H, spec.d
    Lq = spec.n_cur_frames * T_f

    q = _randn_bf16(gen, (B, H, Lq, d))
    k_cache = torch.empty((spec.n_pages, H, T_f, d), dtype=torch.bfloat16)
    v_cache = torch.empty((spec.n_pages, H, T_f, d), dtype=torch.bfloat16)
    # every page of the pool is filled (so a wrong page id changes the answer)
    for p in range(spec.n_pages):
        kp = torch.randn((H, T_f, d), generator=gen, dtype=torch.float32)
        if spec.k_frame_offset_std > 0.0:
            mu = torch.randn((H, 1, d), generator=gen, dtype=torch.float32) * spec.k_frame_offset_std
            kp = kp + mu
        k_cache[p] = kp.to(torch.bfloat16)
        v_cache[p] = _randn_bf16(gen, (H, T_f, d))

    # frame lists: memory (random distinct, unsorted) | window (oldest -> newest) | chunk
    frames: List[List[int]] = []
    if spec.explicit_frames is not None:
        frames = [list(f) for f in spec.explicit_frames]
    else:
        ppc = spec.pages_per_call if spec.pages_per_call is not None else spec.n_pages
        for b in range(B):
            base = b * ppc if spec.pages_per_call is not None else 0
            hi = base + ppc
            cur = list(range(hi - spec.n_cur_frames, hi))
            win = list(range(hi - spec.n_cur_frames - spec.n_win[b], hi - spec.n_cur_frames))
            n_free = ppc - spec.n_cur_frames - spec.n_win[b]
            assert spec.n_mem[b] <= n_free, "not enough pages for the retrieved memory"
            perm = torch.randperm(n_free, generator=gen)[: spec.n_mem[b]]
            mem = [base + int(x) for x in perm]
            frames.append(mem + win + cur)
    frame_off = np.zeros(B + 1, dtype=np.int32)
    for b in range(B):
        frame_off[b + 1] = frame_off[b] + len(frames[b])
    frame_idx = np.asarray([p for f in frames for p in f], dtype=np.int32)

    top_k = np.zeros(B, dtype=np.int32)
    for b in range(B):
        top_k[b] = 0
    prob = Problem(spec, q, k_cache, v_cache, frame_idx, frame_off, top_k)
    for b in range(B):
        top_k[b] = top_k_for(spec, prob.M(b))
    return prob


# --------------------------------------------------------------------------------------
# BASELINE.json configs (seeds, pools, frame lists)
# --------------------------------------------------------------------------------------
def spec_tiny() -> Spec:
    return Spec("tiny", 1001, H=2, d=64, frame_tokens=256, n_cur_frames=1, block=64, n_pages=8,
                n_mem=[2], n_win=[1], top_k=8, explicit_frames=[[0, 3, 6, 7]])


def spec_mid(H: int = 24) -> Spec:
    return Spec("mid", 2002, H=H, d=128, frame_tokens=1560, n_cur_frames=4, block=128, n_pages=64,
                n_mem=[4], n_win=[8], density=Fraction(1, 4))


def spec_long(H: int = 24) -> Spec:
    return Spec("long", 3003, H=H, d=128, frame_tokens=1560, n_cur_frames=4, block=128, n_pages=128,
                n_mem=[16], n_win=[16], density=Fraction(1, 10), k_frame_offset_std=0.5)


def spec_adaptive(H: int = 24) -> Spec:
    return Spec("adaptive", 4004, H=H, d=128, frame_tokens=1560, n_cur_frames=4, block=128,
                n_pages=256, n_mem=[0, 0, 2, 4, 0, 8, 1, 0], n_win=[1, 2, 2, 4, 8, 2, 1, 4],
                density=Fraction(3, 10), pages_per_call=32)


def spec_dense_equivalence(H: int = 24) -> Spec:
    return Spec("dense-equivalence", 5005, H=H, d=128, frame_tokens=1560, n_cur_frames=4, block=128,
                n_pages=64, n_mem=[4], n_win=[8], density=Fraction(1, 1))


def spec_mid3d(H: int = 24) -> Spec:
    """`mid` with the paper's own block geometry: 30 x 52 latent grid, 3-D blocks (4,8,4)."""
    return Spec("mid3d", 6006, H=H, d=128, frame_tokens=1560, n_cur_frames=4, block=128, n_pages=64,
                n_mem=[4], n_win=[8], density=Fraction(1, 4), grid=(30, 52), block3d=(4, 8, 4))


def spec_mid3d448(H: int = 24) -> Spec:
    """`mid` with the paper's second block geometry, (4,4,8) (Matrix-Game-3.0), on the same 30 x 52 grid:
    52 is not a multiple of 8, so every 7th column block is a half-width border block; 30 = 7*4 + 2 leaves a 2-row bottom
    border."""
    return Spec("mid3d448", 8008, H=H, d=128, frame_tokens=1560, n_cur_frames=4, block=128, n_pages=64,
                n_mem=[4], n_win=[8], density=Fraction(1, 4), grid=(30, 52), block3d=(4, 4, 8))


def spec_long3d(H: int = 24) -> Spec:
    """`long` (16 memory + 16 window frames, density 1/10, K offsets) with the paper's 3-D blocks: 416 history blocks."""
    return Spec("long3d", 7007, H=H, d=128, frame_tokens=1560, n_cur_frames=4, block=128, n_pages=128,
                n_mem=[16], n_win=[16], density=Fraction(1, 10), k_frame_offset_std=0.5, grid=(30, 52), block3d=(4, 8, 4))


def spec_by_name(name: str, H: Optional[int] = None) -> Spec:
    table = {"tiny": spec_tiny, "mid": spec_mid, "long": spec_long, "adaptive": spec_adaptive,
             "dense-equivalence": spec_dense_equivalence, "mid3d": spec_mid3d, "long3d": spec_long3d,
             "mid3d448": spec_mid3d448}
    fn = table[name]
    if name == "tiny" or H is None:
        return fn()
    return fn(H)


# Reduced shapes for element-by-element parity: the oracle finishes them in seconds, yet they
# keep what makes the full configs awkward: T_f not a multiple of the block (blocks straddle
# frames), ragged history tail, ragged chunk tail, several query tiles, unsorted memory pages.
def spec_small(name: str = "small", seed: int = 7007, H: int = 2, d: int = 128, block: int = 128,
               frame_tokens: int = 200, n_cur_frames: int = 3, n_pages: int = 12,
               n_mem=(2,), n_win=(3,), density=Fraction(1, 2), top_k=None,
               k_frame_offset_std: float = 0.0, pages_per_call=None, grid=None, block3d=None) -> Spec:
    return Spec(name, seed, H=H, d=d, frame_tokens=frame_tokens, n_cur_frames=n_cur_frames,
                block=block, n_pages=n_pages, n_mem=list(n_mem), n_win=list(n_win),
                density=None if top_k is not None else density, top_k=top_k,
                k_frame_offset_std=k_frame_offset_std, pages_per_call=pages_per_call, grid=grid, block3d=block3d)


def effective_flops(prob: Problem, sel_idx_per_call, sel_cnt_per_call) -> int:
    """4*d*sum_{b,h,i} valid_q(i) * (Lc + sum_{m in I_i} valid_k(m)).
    Pure integer bookkeeping over an ALREADY COMPUTED mask; no method arithmetic."""
    s = prob.spec
    Lc = s.n_cur_frames * s.frame_tokens
    vq = prob.block_sizes(s.n_cur_frames)                      # [Nqb]
    total = 0
    for b in range(prob.B):
        vk = prob.block_sizes(prob.n_hist_frames(b))           # [M_b]
        idx = np.asarray(sel_idx_per_call[b])                  # [H, Nqb, >=k]
        cnt = np.asarray(sel_cnt_per_call[b])                  # [H, Nqb]
        kk = idx.shape[-1]
        live = np.arange(kk)[None, None, :] < cnt[:, :, None]
        tok = np.where(live, vk[np.clip(idx, 0, max(len(vk) - 1, 0))] if len(vk) else 0, 0).sum(axis=-1)   # [H, Nqb]
        total += int((4 * s.d * vq[None, :] * (tok + Lc)).sum())
    return total
