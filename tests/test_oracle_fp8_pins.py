"""Pins for oracle/li_fp8_oracle.py (fp8 E4M3 K/V pages), CPU only.  Each test checks the oracle against
something that is not itself: torch's float8_e4m3fn type (a library implementation of the same OCP format), hand-worked
code points / ties / saturation, an exact-arithmetic invariance, and the bf16 oracle where fp8 loses nothing."""
import numpy as np
import pytest
import torch

from oracle import li_fp8_oracle as F
from oracle import li_oracle as O

RNG = np.random.default_rng(2605)


def test_decode_table_matches_library_type_for_all_256_codes():
    codes = np.arange(256, dtype=np.uint8)
    ref = torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    got = F.e4m3_decode(codes)
    assert np.isnan(got[0x7F]) and np.isnan(got[0xFF]) and np.isnan(ref[0x7F]) and np.isnan(ref[0xFF])
    ok = ~np.isnan(ref)
    np.testing.assert_array_equal(got[ok], ref[ok])


def test_hand_worked_code_points():
    """From the format definition: bias 7, 3 mantissa bits, subnormals (m/8) * 2^-6, max finite 1.75 * 2^8 = 448."""
    dec = F.e4m3_decode
    assert dec(np.uint8(0x00)) == 0.0 and dec(np.uint8(0x80)) == 0.0 and np.signbit(dec(np.uint8(0x80)))
    assert dec(np.uint8(0x01)) == 2.0 ** -9                     # smallest subnormal
    assert dec(np.uint8(0x07)) == 7 * 2.0 ** -9                 # largest subnormal
    assert dec(np.uint8(0x08)) == 2.0 ** -6                     # smallest normal
    assert dec(np.uint8(0x38)) == 1.0 and dec(np.uint8(0x39)) == 1.125 and dec(np.uint8(0x40)) == 2.0
    assert dec(np.uint8(0x7E)) == 448.0 and dec(np.uint8(0xFE)) == -448.0
    assert dec(np.uint8(0xB8)) == -1.0


def test_every_finite_code_round_trips_exactly():
    codes = np.asarray([c for c in range(256) if c not in (0x7F, 0xFF)], dtype=np.uint8)
    back = F.e4m3_encode(F.e4m3_decode(codes))
    np.testing.assert_array_equal(back, codes)                  # including -0 -> 0x80


def test_ties_to_even_subnormals_and_saturation_by_hand():
    enc = lambda v: int(F.e4m3_encode(np.asarray(v, dtype=np.float64)))
    assert enc(1.0625) == 0x38          # half-way 1.0 (m=0) | 1.125 (m=1) -> even mantissa -> 1.0
    assert enc(1.1875) == 0x3A          # half-way 1.125 (m=1) | 1.25 (m=2) -> 1.25
    assert enc(1.0626) == 0x39 and enc(1.1874) == 0x39
    assert enc(1.9375) == 0x40          # half-way 1.875 (m=7, e=7) | 2.0 (m=0, e=8): the even code is 2.0
    assert enc(2.0 ** -10) == 0x00      # half-way 0 | 2^-9 -> 0
    assert enc(3 * 2.0 ** -10) == 0x02  # half-way 2^-9 (m=1) | 2^-8 (m=2) -> m=2
    assert enc(-3 * 2.0 ** -10) == 0x82
    assert enc(448.0) == 0x7E and enc(463.9) == 0x7E and enc(464.0) == 0x7E and enc(1e9) == 0x7E and enc(-1e9) == 0xFE
    assert enc(np.inf) == 0x7E and enc(-np.inf) == 0xFE and enc(np.nan) == 0x7F
    assert enc(0.0) == 0x00 and enc(-0.0) == 0x80


def test_encode_matches_library_conversion_inside_the_finite_range():
    """torch's float32 -> float8_e4m3fn conversion is round-to-nearest-even; compared on random values and on every
    half-way point between neighbouring code points (|x| <= 448: beyond it torch does not saturate)."""
    table = F.e4m3_table()[:0x7F]
    mids = (table[:-1] + table[1:]) / 2
    x = np.concatenate([RNG.uniform(-448, 448, 20000), RNG.normal(0, 1, 20000), RNG.normal(0, 0.01, 5000), mids, -mids,
                        table, -table]).astype(np.float32)
    ref = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = F.e4m3_encode(x.astype(np.float64))
    np.testing.assert_array_equal(got, ref)


def small_problem(H=2, d=16, T_f=24, n_pages=7, frames=(5, 1, 4, 2, 6), n_cur=2, block=16):
    g = torch.Generator().manual_seed(88)
    q = torch.randn((1, H, n_cur * T_f, d), generator=g).to(torch.bfloat16)
    k = torch.randn((n_pages, H, T_f, d), generator=g).to(torch.bfloat16)
    v = torch.randn((n_pages, H, T_f, d), generator=g).to(torch.bfloat16)
    u16 = lambda t: t.view(torch.int16).numpy().view(np.uint16)
    fi, fo = np.asarray(frames, np.int32), np.asarray([0, len(frames)], np.int32)
    return u16(q), O.widen(u16(k)), O.widen(u16(v)), fi, fo, n_cur, block


def test_quantise_on_write_and_dequantise():
    q, k, v, fi, fo, n_cur, block = small_problem()
    ks = np.asarray([0.011, 0.02], np.float32)
    codes = F.quantize(k, ks, head_axis=1)
    back = F.dequantize(codes, ks, head_axis=1)
    # relative error of a normal code point is at most half an ulp = 2^-4; absolute error for subnormals 2^-10 * scale
    err = np.abs(back - k)
    bound = np.maximum(np.abs(k) * 2.0 ** -4, 2.0 ** -10 * ks.astype(np.float64).reshape(1, -1, 1, 1)) * (1 + 1e-6)
    assert (err <= bound).all()
    # an explicit element: value / scale rounded in fp32, then to the nearest code point
    x = np.float32(k[3, 1, 5, 7]) / ks[1]
    assert codes[3, 1, 5, 7] == F.e4m3_encode(np.float64(x))


def test_scale_invariance_of_scores_and_attention():
    """decode(code) * (c * scale) == c * (decode(code) * scale): doubling k_scale equals doubling softmax_scale (powers of
    two are exact), and doubling v_scale doubles the output."""
    q, k, v, fi, fo, n_cur, block = small_problem()
    ks, vs = np.asarray([0.0125, 0.02], np.float32), np.asarray([0.015, 0.01], np.float32)
    kc, vc = F.quantize(k, ks, 1), F.quantize(v, vs, 1)
    sel, sc = F.block_select_fp8(q, kc, ks, fi, fo, n_cur, block, block, [3])
    sel2, sc2 = F.block_select_fp8(q, kc, 2 * ks, fi, fo, n_cur, block, block, [3])
    np.testing.assert_array_equal(sel[0], sel2[0])
    np.testing.assert_array_equal(sc2[0], 2 * sc[0])
    o1, l1 = F.sparse_attn_fp8(q, kc, vc, 2 * ks, vs, fi, fo, n_cur, block, block, sel, softmax_scale=0.125)
    o2, l2 = F.sparse_attn_fp8(q, kc, vc, ks, 2 * vs, fi, fo, n_cur, block, block, sel, softmax_scale=0.25)
    np.testing.assert_allclose(2 * o1, o2, rtol=0, atol=1e-6)
    np.testing.assert_allclose(l1, l2, rtol=0, atol=1e-6)


def test_reproduces_the_bf16_oracle_when_nothing_is_lost():
    """Values on the e4m3 grid (3 mantissa bits, here {0, +-0.25 .. +-3.5}) with scale 1 survive quantisation exactly, and
    query rows whose largest entry is 3.5 keep their values under the per-row scale 3.5/448 = 2^-7: the fp8 oracle must
    then equal li_oracle.py on the bf16 tensors bit for bit."""
    g = np.random.default_rng(7)
    grid = np.asarray([0.0, 0.25, 0.5, 0.75, 1.0, 1.25, 1.5, 1.75, 2.0, 2.5, 3.0, 3.5])
    H, d, T_f, n_pages, n_cur, block = 2, 16, 24, 6, 2, 16

    def draw(shape):
        x = g.choice(grid, size=shape) * g.choice([-1.0, 1.0], size=shape)
        return x

    q = draw((1, H, n_cur * T_f, d))
    q[..., 0] = 3.5                                              # every row's amax is 3.5 -> row scale exactly 2^-7
    k, v = draw((n_pages, H, T_f, d)), draw((n_pages, H, T_f, d))
    to_bits = lambda x: torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    fi, fo = np.asarray([4, 0, 3, 1, 5], np.int32), np.asarray([0, 5], np.int32)
    one = np.ones(H, np.float32)
    kc, vc = F.quantize(k, one, 1), F.quantize(v, one, 1)
    np.testing.assert_array_equal(F.dequantize(kc, one, 1), k)
    np.testing.assert_array_equal(F.quantize_query_rows(to_bits(q)), q)
    sel, sc = F.block_select_fp8(to_bits(q), kc, one, fi, fo, n_cur, block, block, [2])
    sel_ref, sc_ref = O.block_select(to_bits(q), to_bits(k), fi, fo, n_cur, block, block, [2])
    np.testing.assert_array_equal(sel[0], sel_ref[0])
    np.testing.assert_array_equal(sc[0], sc_ref[0])
    o, lse = F.sparse_attn_fp8(to_bits(q), kc, vc, one, one, fi, fo, n_cur, block, block, sel)
    o_ref, lse_ref = O.sparse_attn(to_bits(q), to_bits(k), to_bits(v), fi, fo, n_cur, block, block, sel_ref)
    np.testing.assert_array_equal(o, o_ref)
    np.testing.assert_array_equal(lse, lse_ref)


def test_query_rows_are_quantised_per_row():
    q = np.zeros((1, 1, 3, 8), np.float32)
    q[0, 0, 0] = [448, 1, -2, 0.3, 0, 0, 0, 0]                   # scale 1: 0.3 -> nearest code point 0.3125
    q[0, 0, 1] = [0.07, -0.0101, 0, 0, 0, 0, 0, 0]
    got = F.quantize_query_rows(q)
    assert got[0, 0, 0].tolist() == [448.0, 1.0, -2.0, 0.3125, 0, 0, 0, 0]
    qs = np.float32(0.07) / np.float32(448)
    assert got[0, 0, 1, 0] == 448.0 * np.float64(qs)
    x = np.float32(-0.0101) / qs                                 # -64.64 -> code points 60 | 64 | 72: nearest 64
    assert got[0, 0, 1, 1] == -64.0 * np.float64(qs) and abs(float(x) + 64.64) < 0.01
    assert (got[0, 0, 2] == 0).all()                             # a zero row stays zero (scale 1)
