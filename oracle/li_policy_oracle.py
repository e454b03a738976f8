"""CPU ORACLE for Light Interaction's adaptive context management (Eq. 1-4) and the frame-list
reconstruction it drives (Fig. 2a; BASELINE.json north_star (b):  memory | temporal window | current chunk).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as li_oracle.py): only `tests/` may import it; it shares no code
with the CUDA path.

  Eq. 1  D_t = MSE(z_{t-1}, z_{t-2}), averaged over all latent dimensions;
  Eq. 2  Dbar_t = alpha D_t + (1 - alpha) Dbar_{t-1}, initialised by the first valid D_t;
  Eq. 3  L_t = clip([L_m kappa / (Dbar_t + kappa)], 1, L_m).  The bracket is garbled in the source ("|.|"):
                       floor and round-to-nearest are both offered (reading c18), `rounding` selects;
  Eq. 4  max_j S_pose(t, j) < tau_pose  =>  pure exploration: the retrieved memory is discarded;
  frame list           [retrieved memory pages, if kept] + [the L_t most recent window pages] + [current chunk pages].

Arithmetic: fp64 (numpy), inputs widened exactly.  Eq. 3 turns a floating-point value into an integer; both sides must
take that decision in the same precision, so `window_length` takes the dtype the decision is evaluated in (fp64 by
default; the parity test passes float32 = the kernel's, with the operation order written below).
Pins: tests/test_oracle_policy_pins.py (hand-worked numbers, closed forms, limits, monotonicity, strictness of Eq. 4).
"""
from __future__ import annotations

from typing import Optional, Sequence, Tuple

import numpy as np


def latent_mse(z_prev1: np.ndarray, z_prev2: np.ndarray) -> float:
    """Eq. 1: mean over ALL latent dimensions of the squared difference of the two most recent stable units."""
    a = np.asarray(z_prev1, dtype=np.float64).ravel()
    b = np.asarray(z_prev2, dtype=np.float64).ravel()
    assert a.shape == b.shape and a.size > 0
    return float(((a - b) ** 2).sum() / a.size)


def ema_update(D_t: float, D_bar_prev: Optional[float], alpha: float) -> float:
    """Eq. 2: exponential moving average; `D_bar_prev is None` = no valid D yet -> initialised by D_t."""
    assert 0.0 < alpha <= 1.0
    if D_bar_prev is None:
        return float(D_t)
    return float(alpha * D_t + (1.0 - alpha) * D_bar_prev)


def window_length(D_bar: float, kappa: float, L_m: int, rounding: str = "floor", dtype=np.float64) -> int:
    """Eq. 3: L_t = clip([L_m * kappa / (Dbar + kappa)], 1, L_m), evaluated in `dtype` in exactly this
    order: (L_m * kappa) / (Dbar + kappa), then floor or round-half-to-even, then the clip."""
    assert kappa > 0 and L_m >= 1 and rounding in ("floor", "nearest")
    t = dtype(L_m)
    x = (t * dtype(kappa)) / (dtype(D_bar) + dtype(kappa))
    v = np.floor(x) if rounding == "floor" else np.rint(x)
    return int(min(max(int(v), 1), L_m))


def keep_memory(s_pose: Sequence[float], tau_pose: float) -> bool:
    """Eq. 4: the retrieved memory is discarded iff max_j S_pose(t, j) < tau_pose (strict).  Without any
    candidate there is nothing to keep."""
    s = np.asarray(s_pose, dtype=np.float64)
    if s.size == 0:
        return False
    return not (float(s.max()) < float(tau_pose))


def reconstruct_frame_list(mem_pages: Sequence[int], win_pages: Sequence[int], cur_pages: Sequence[int], L_t: int,
                           keep: bool) -> np.ndarray:
    """The reconstructed context as a page list: retrieved memory (if kept) | the L_t most recent units of the temporal
    window (win_pages is ordered oldest -> newest; fewer than L_t available: all of them) | the current chunk."""
    mem = list(mem_pages) if keep else []
    n = min(int(L_t), len(win_pages))
    win = list(win_pages)[len(win_pages) - n:] if n > 0 else []
    return np.asarray(mem + win + list(cur_pages), dtype=np.int32)


def context_policy(z_prev1, z_prev2, D_bar_prev: Optional[float], alpha: float, kappa: float, L_m: int, s_pose, tau_pose: float,
                   mem_pages, win_pages, cur_pages, rounding: str = "floor") -> Tuple[float, float, int, bool, np.ndarray]:
    """Eq. 1-4 in the paper's order, then the page list.  -> (D_t, Dbar_t, L_t, keep_memory, frame_idx)."""
    D_t = latent_mse(z_prev1, z_prev2)
    D_bar = ema_update(D_t, D_bar_prev, alpha)
    L_t = window_length(D_bar, kappa, L_m, rounding)
    keep = keep_memory(s_pose, tau_pose)
    return D_t, D_bar, L_t, keep, reconstruct_frame_list(mem_pages, win_pages, cur_pages, L_t, keep)
