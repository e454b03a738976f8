"""GPU parity for the paper's 3-D block tiling (B_t,B_h,B_w) against oracle/li_oracle.py *_3d."""
from fractions import Fraction

import numpy as np
import pytest
import torch

import li_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    from tests import parity_util
    return parity_util


def small3d(name, grid, block3d, n_cur, n_mem, n_win, H=2, d=128, density=Fraction(1, 2), n_pages=14, **kw):
    gh, gw = grid
    bt, bh, bw = block3d
    return W.spec_small(name=name, H=H, d=d, block=bt * bh * bw, frame_tokens=gh * gw, n_cur_frames=n_cur,
                        n_pages=n_pages, n_mem=n_mem, n_win=n_win, density=density, grid=grid, block3d=block3d, **kw)


@pytest.mark.parametrize("grid,block3d,n_cur,n_hist", [((30, 52), (4, 8, 4), 4, (2, 4)),     # paper geometry, partial rows
                                                        ((10, 16), (4, 4, 8), 4, (3, 3)),     # Matrix-Game block shape
                                                        ((12, 8), (2, 8, 4), 2, (2, 3)),      # 64-token blocks, partial group
                                                        ((6, 8), (4, 8, 4), 3, (1, 4))])      # grid lower than a block, partial groups
def test_select_3d(P, grid, block3d, n_cur, n_hist):
    spec = small3d(f"s3d-{grid}-{block3d}", grid, block3d, n_cur, (n_hist[0],), (n_hist[1],))
    prob = W.build(spec)
    excused = P.select_parity(prob)
    print(f"{spec.name}: M={prob.M(0)} Nqb={prob.Nqb} k={int(prob.top_k[0])} excused={excused}")


@pytest.mark.parametrize("grid,block3d,n_cur,n_hist,d", [((30, 52), (4, 8, 4), 4, (2, 4), 128),   # paper geometry: rows 24..29 partial
                                                          ((10, 16), (4, 4, 8), 4, (3, 3), 128),   # (4,4,8), partial group (6 frames)
                                                          ((12, 8), (2, 8, 4), 2, (2, 3), 64),     # 64-token blocks, d=64
                                                          ((6, 8), (4, 8, 4), 3, (1, 4), 128)])    # partial chunk group (3 of 4 frames)
def test_full_parity_3d(P, grid, block3d, n_cur, n_hist, d):
    """li_block_select + li_sparse_attn with 3-D blocks, element by element against the oracle: 5-D TMA boxes, zero
    filled grid rows / missing frames masked out, outputs scattered back to linear token order."""
    H = 1 if grid == (30, 52) else 2
    spec = small3d(f"f3d-{grid}-{block3d}", grid, block3d, n_cur, (n_hist[0],), (n_hist[1],), H=H, d=d)
    prob = W.build(spec)
    excused, mx, mean = P.full_parity(prob)
    print(f"{spec.name}: M={prob.M(0)} Nqb={prob.Nqb} k={int(prob.top_k[0])} excused={excused} max-abs={mx:.3g} mean-abs={mean:.3g}")


def test_3d_dense_and_chunk_only(P):
    """r = 1 -> dense attention over the whole context (torch SDPA); k = 0 -> chunk-only attention."""
    for density, name in ((Fraction(1, 1), "dense"), (None, "k0")):
        spec = small3d(f"f3d-{name}", (10, 16), (4, 8, 4), 4, (1,), (2,), density=density or Fraction(1, 2),
                       **({"top_k": 0} if density is None else {}))
        prob = W.build(spec)
        ctx, buf = P.run_gpu(prob)
        frames = prob.frame_idx if density is not None else prob.frame_idx[-4:]
        K = torch.cat([prob.k_cache[int(p)] for p in frames], dim=1).float()
        V = torch.cat([prob.v_cache[int(p)] for p in frames], dim=1).float()
        ref = torch.nn.functional.scaled_dot_product_attention(prob.q[0].float(), K, V)
        diff = (buf.o[0].float().cpu() - ref).abs()
        assert torch.isfinite(buf.o.float()).all() and diff.max() <= P.MAX_ABS and diff.mean() <= P.MEAN_ABS
