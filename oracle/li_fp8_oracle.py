"""CPU ORACLE for the fp8 K/V-page variant of the Light Interaction sparse-attention path.

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as li_oracle.py): only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s oracle legs may import it; it shares no code with the CUDA path.

The paper states no numeric precision for its cache (PAPER.md:170 gives hardware and ratios only), so the storage format
is a reading (DESIGN.md c20): K and V pages are held as OCP FP8 E4M3 ("e4m3fn": 1 sign, 4 exponent bits with bias 7,
3 mantissa bits, no infinities, the single NaN pattern S.1111.111, largest finite value 448) together with one fp32
scale per head, value = decode(code) * scale[h]; a page is quantised once, when it is written
(code = encode(value / scale[h]), round to nearest even, saturating at +-448).  What the path then computes is the
SAME method as li_oracle.py (Eq. 9-11 + softmax attention) on the dequantised cache, with every query row q_u
replaced by its own e4m3 image: qs_u = max_c |q_u[c]| / 448 (fp32; 1 if the row is zero), q^_u = decode(encode(q_u /
qs_u)) * qs_u, because the fp8 tensor-core MMA takes both operands in 8 bits.  Block selection (Eq. 9-10) pools the
unquantised Q and the dequantised K.  The attention probabilities are an internal quantity of the kernel (it rounds
them to e4m3 before the second MMA); the oracle keeps them exact and the parity tolerance accounts for that rounding
(DESIGN.md c20).

encode/decode are written from the format definition (a table of the 256 code points; nearest code point, ties to the
even mantissa).  Pins (tests/test_oracle_fp8_pins.py): the decode table against torch.float8_e4m3fn (a library type)
for all 256 codes; exact round trip of every finite code; hand-worked ties, subnormals and saturation; agreement with
torch's own float32 -> float8_e4m3fn conversion on random and half-way inputs inside the finite range; scale invariance
(k_scale * c == softmax_scale * c); reproduction of li_oracle.py when every value is fp8-representable.
"""
from __future__ import annotations

from typing import Sequence

import numpy as np

from oracle import li_oracle as O

E4M3_MAX = 448.0


def e4m3_table() -> np.ndarray:
    """value of every code point 0..255 (fp64); the two NaN patterns 0x7f / 0xff are NaN."""
    out = np.zeros(256, dtype=np.float64)
    for code in range(256):
        sign = -1.0 if code & 0x80 else 1.0
        e, m = (code >> 3) & 0xF, code & 0x7
        if e == 0xF and m == 0x7:
            out[code] = np.nan
        elif e == 0:
            out[code] = sign * (m / 8.0) * 2.0 ** (-6)            # subnormal: no implicit one
        else:
            out[code] = sign * (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return out


_TABLE = e4m3_table()
_POS = _TABLE[:0x7F]                                                # codes 0x00..0x7e: ascending, 0 .. 448


def e4m3_decode(codes: np.ndarray) -> np.ndarray:
    return _TABLE[np.asarray(codes, dtype=np.uint8)]


def e4m3_encode(x: np.ndarray) -> np.ndarray:
    """Nearest code point, ties to the even mantissa code, magnitudes beyond 448 saturate to +-448, NaN -> 0x7f.
    (The semantics of PTX cvt.rn.satfinite.e4m3x2.f32.)"""
    x = np.asarray(x, dtype=np.float64)
    mag = np.minimum(np.abs(x), E4M3_MAX)
    hi = np.searchsorted(_POS, mag, side="left")                    # first code point >= mag
    hi = np.clip(hi, 0, len(_POS) - 1)
    lo = np.maximum(hi - 1, 0)
    d_lo, d_hi = mag - _POS[lo], _POS[hi] - mag
    pick_hi = (d_hi < d_lo) | ((d_hi == d_lo) & (hi % 2 == 0))     # tie: the code with an even mantissa (even code)
    code = np.where(pick_hi, hi, lo).astype(np.uint8)
    code = np.where(np.signbit(x), code | 0x80, code).astype(np.uint8)
    return np.where(np.isnan(x), np.uint8(0x7F), code).astype(np.uint8)


def quantize(values: np.ndarray, scale_per_head: Sequence[float], head_axis: int) -> np.ndarray:
    """Quantise-on-write: code = encode(value / scale[h]) with the division taken in fp32 (the kernel's precision: a
    floating-point value decides an integer code, both sides decide in fp32).  values: float array (bf16 values widened)."""
    v = np.asarray(values, dtype=np.float32)
    shape = [1] * v.ndim
    shape[head_axis] = -1
    s = np.asarray(scale_per_head, dtype=np.float32).reshape(shape)
    return e4m3_encode((v / s).astype(np.float64))


def dequantize(codes: np.ndarray, scale_per_head: Sequence[float], head_axis: int) -> np.ndarray:
    shape = [1] * np.ndim(codes)
    shape[head_axis] = -1
    return e4m3_decode(codes) * np.asarray(scale_per_head, dtype=np.float32).astype(np.float64).reshape(shape)


def quantize_query_rows(q: np.ndarray) -> np.ndarray:
    """q: bf16 bit patterns or floats [..., d] -> the e4m3 image of every row, fp64: qs = amax / 448 in fp32 (1 for a zero
    row), code = encode(q / qs) with the division in fp32, value = decode(code) * qs."""
    qf = O.widen(q).astype(np.float32)
    amax = np.abs(qf).max(axis=-1, keepdims=True)
    qs = np.where(amax > 0, amax / np.float32(E4M3_MAX), np.float32(1.0)).astype(np.float32)
    codes = e4m3_encode((qf / qs).astype(np.float64))
    return e4m3_decode(codes) * qs.astype(np.float64)


def block_select_fp8(q, k_codes, k_scale, frame_idx, frame_off, n_cur_frames: int, block_q: int, block_k: int, top_k):
    """Eq. 9-10 on the dequantised K cache (k_codes uint8 [n_pages,H,T_f,d], k_scale fp32 [H]); Q is pooled unquantised."""
    return O.block_select(q, dequantize(k_codes, k_scale, 1), frame_idx, frame_off, n_cur_frames, block_q, block_k, top_k)


def sparse_attn_fp8(q, k_codes, v_codes, k_scale, v_scale, frame_idx, frame_off, n_cur_frames: int, block_q: int,
                    block_k: int, sel_idx, softmax_scale: float = 0.0, tiles=None):
    """Eq. 11 + softmax attention over the dequantised cache, every query row replaced by its e4m3 image."""
    return O.sparse_attn(quantize_query_rows(q), dequantize(k_codes, k_scale, 1), dequantize(v_codes, v_scale, 1),
                         frame_idx, frame_off, n_cur_frames, block_q, block_k, sel_idx, softmax_scale=softmax_scale,
                         tiles=tiles)
