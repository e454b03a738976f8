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
