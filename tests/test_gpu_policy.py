"""GPU parity of li_context_policy (Eq. 1-4 + frame-list reconstruction, include/li.h) against
oracle/li_policy_oracle.py, through the C-ABI binding."""
from fractions import Fraction

import numpy as np
import pytest
import torch

import li_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import paper_2605_31158_b200 as li
    from oracle import li_policy_oracle as PO
    return li, PO


def _dev(x, dtype):
    return torch.as_tensor(np.asarray(x), dtype=dtype).cuda()


def run_policy(li, z1, z2, ema, alpha, kappa, L_max, s_pose, tau, mem, win, cur, nearest=False, cap=None):
    cap = cap if cap is not None else len(mem) + min(L_max, len(win)) + len(cur)
    out = torch.full((cap + 4,), -7, dtype=torch.int32, device="cuda")
    res = torch.zeros(24, dtype=torch.uint8, device="cuda")
    ws = torch.empty(li.lib().li_policy_workspace_bytes(), dtype=torch.uint8, device="cuda")
    li.li_context_policy(z1, z2, ema, alpha, kappa, L_max, _dev(s_pose, torch.float32) if len(s_pose) else None, tau,
                         _dev(mem, torch.int32) if len(mem) else None, _dev(win, torch.int32) if len(win) else None,
                         _dev(cur, torch.int32), out, res, ws, round_nearest=nearest)
    torch.cuda.synchronize()
    return li.policy_result(res), out.cpu().numpy()


@pytest.mark.parametrize("dtype,n", [(torch.float32, 16 * 4 * 60 * 104), (torch.bfloat16, 16 * 4 * 60 * 104 + 5),
                                     (torch.float32, 3), (torch.bfloat16, 4096 * 1024 + 1)])
@pytest.mark.parametrize("nearest", [False, True])
def test_policy_sequence_matches_oracle(env, dtype, n, nearest):
    """Three consecutive chunks: D_t (Eq. 1) of ragged-size latents, the EMA state carried on the device (Eq. 2, first
    call initialises), the window length (Eq. 3, decided in fp32 on both sides), the gate (Eq. 4) and the page list."""
    li, PO = env
    g = torch.Generator().manual_seed(1234 + n % 97)
    ema = torch.zeros(2, dtype=torch.float32, device="cuda")
    alpha, kappa, L_max, tau = 0.3, 0.02, 12, 0.45
    mem, win, cur = [50, 3, 17], list(range(100, 120)), [7, 8, 9, 10]
    Db_ref = None
    for step, (amp, s_pose) in enumerate([(0.05, [0.2, 0.6, 0.1]), (0.3, [0.1, 0.44999, 0.3]), (0.11, [0.45])]):
        z2 = torch.randn(n, generator=g).to(dtype)
        z1 = (z2.float() + amp * torch.randn(n, generator=g)).to(dtype)
        r, out = run_policy(li, z1.cuda(), z2.cuda(), ema, alpha, kappa, L_max, s_pose, tau, mem, win, cur, nearest)
        D_ref = PO.latent_mse(z1.float().numpy(), z2.float().numpy())
        Db_ref = PO.ema_update(D_ref, Db_ref, alpha)
        assert r.D_t == pytest.approx(D_ref, rel=3e-6), "Eq. 1"
        assert r.D_bar == pytest.approx(Db_ref, rel=1e-5), "Eq. 2"
        assert ema.cpu().tolist() == [r.D_bar, 1.0]
        rounding = "nearest" if nearest else "floor"
        # Eq. 3 decides an integer from a float.  The seeded inputs keep L_m kappa / (Dbar + kappa) at least 3.9e-3 away
        # from every floor / round-half boundary (checked here), a thousand times the fp32-vs-fp64 difference of that
        # quotient, so the INDEPENDENT fp64 decision of the oracle must be reproduced, unconditionally ...
        x = L_max * kappa / (Db_ref + kappa)
        assert abs(x - np.round(x * 2) / 2) > 1e-3, "test input sits on a rounding boundary: pick another seed"
        assert r.L_t == PO.window_length(Db_ref, kappa, L_max, rounding)
        # ... and, as documented in li.h (operation order is part of the interface), the fp32 evaluation of the kernel's
        # own Dbar as well
        assert r.L_t == PO.window_length(r.D_bar, kappa, L_max, rounding, np.float32)
        keep = PO.keep_memory(s_pose, tau)
        assert bool(r.keep_memory) == keep, "Eq. 4"
        want = PO.reconstruct_frame_list(mem, win, cur, r.L_t, keep)
        assert r.n_frames == len(want) and r.n_hist_frames == len(want) - len(cur)
        np.testing.assert_array_equal(out[:r.n_frames], want)
        assert (out[r.n_frames:] == -7).all(), "entries past n_frames must stay untouched"


@pytest.mark.parametrize("c,kappa,L_max,L_floor,L_nearest", [
    (0.5, 0.25, 8, 4, 4),       # D = 1/4:  8 * 1/4 / (1/4 + 1/4)   = 4       exactly on an integer
    (0.25, 0.25, 10, 8, 8),     # D = 1/16: 10 * 1/4 / (1/16 + 1/4) = 8       exactly on an integer
    (0.5, 0.25, 5, 2, 2),       # D = 1/4:  5/4 / (1/2)             = 2.5     half-way: floor 2, nearest-even 2
    (0.5, 0.25, 7, 3, 4),       # D = 1/4:  7/4 / (1/2)             = 3.5     half-way: floor 3, nearest-even 4
    (1.0, 0.5, 3, 1, 1),        # D = 1:    3/2 / (3/2)             = 1       lower clip reached exactly
    (0.0, 0.125, 6, 6, 6),      # D = 0:    6/8 / (1/8)             = 6 = L_m upper clip reached exactly
    (2.0, 0.5, 16, 1, 2),       # D = 4:    8 / 4.5 = 1.777...      floor 1, nearest 2 (not a boundary)
])
def test_policy_window_length_on_exact_boundaries(env, c, kappa, L_max, L_floor, L_nearest):
    """Eq. 3 on rounding boundaries whose answer is fixed by hand: z_{t-1} - z_{t-2} = c everywhere gives D_t = c^2 exactly
    (c, c^2, kappa and L_m kappa are dyadic rationals, every fp32 and fp64 operation on them is exact), so
    L_m kappa / (D + kappa) lands exactly on an integer or on a half: the expected L_t is the one written in the
    parameter list, for both readings of the garbled bracket (DESIGN.md c18)."""
    li, PO = env
    n = 4096 + 24
    z2 = torch.full((n,), 0.75).cuda()
    z1 = torch.full((n,), 0.75 + c).cuda()
    for nearest, want in ((False, L_floor), (True, L_nearest)):
        ema = torch.zeros(2, dtype=torch.float32, device="cuda")
        r, out = run_policy(li, z1, z2, ema, 1.0, kappa, L_max, [1.0], 0.5, [3], list(range(40, 60)), [7], nearest)
        assert r.D_t == c * c and r.D_bar == c * c
        assert r.L_t == want, (nearest, r.L_t, want)
        assert r.n_frames == 1 + want + 1 and out[1:1 + want].tolist() == list(range(60 - want, 60))
        assert PO.window_length(c * c, kappa, L_max, "nearest" if nearest else "floor") == want   # the oracle agrees by hand too


def test_policy_ema_on_exact_values(env):
    """Eq. 2 then Eq. 3 with dyadic values: D_1 = 1/4 initialises the EMA; D_2 = 1, alpha = 1/2 -> Dbar = 5/8 exactly;
    kappa = 3/8, L_m = 8 -> 3 / 1 = 3 exactly."""
    li, PO = env
    n = 10007
    ema = torch.zeros(2, dtype=torch.float32, device="cuda")
    z2 = torch.zeros(n).cuda()
    r, _ = run_policy(li, torch.full((n,), 0.5).cuda(), z2, ema, 0.5, 0.375, 8, [], 0.0, [], list(range(8)), [9])
    assert (r.D_t, r.D_bar, r.L_t) == (0.25, 0.25, 4)                # 3 / (5/8) = 4.8 -> floor 4
    r, _ = run_policy(li, torch.full((n,), 1.0).cuda(), z2, ema, 0.5, 0.375, 8, [], 0.0, [], list(range(8)), [9])
    assert (r.D_t, r.D_bar, r.L_t) == (1.0, 0.625, 3)


def test_policy_limits(env):
    """Identical latents -> D = 0 -> whole budget; huge dynamics -> L_t = 1; max == tau keeps the memory (strict <);
    no candidates, no memory, short window."""
    li, PO = env
    z = torch.randn(10000).cuda()
    ema = torch.zeros(2, dtype=torch.float32, device="cuda")
    r, out = run_policy(li, z, z.clone(), ema, 1.0, 0.01, 8, [0.7], 0.7, [5], [1, 2, 3], [9])
    assert (r.D_t, r.L_t, r.keep_memory) == (0.0, 8, 1)
    np.testing.assert_array_equal(out[:r.n_frames], [5, 1, 2, 3, 9])          # only 3 window pages exist
    r, out = run_policy(li, z, z + 100.0, ema, 1.0, 0.01, 8, [], 0.7, [5], [1, 2, 3], [9])
    assert r.D_t == pytest.approx(1e4, rel=1e-5) and r.L_t == 1 and r.keep_memory == 0
    np.testing.assert_array_equal(out[:r.n_frames], [3, 9])
    r, out = run_policy(li, z, z.clone(), ema, 0.5, 0.01, 4, [0.1], 0.7, [], [], [9, 11])
    assert r.D_bar == pytest.approx(0.5 * 1e4, rel=1e-5) and r.n_hist_frames == 0
    np.testing.assert_array_equal(out[:r.n_frames], [9, 11])


def test_policy_output_drives_the_attention_path(env):
    """The device-side frame list produced by li_context_policy is consumed in place by li_block_select /
    li_sparse_attn: with a window of 3 and the memory kept it reproduces the workload's list, and the outputs are
    bit-identical to the run on the uploaded list."""
    li, PO = env
    from tests import parity_util as P
    spec = W.spec_small(name="small-policy", H=2, d=128, block=128, frame_tokens=200, n_cur_frames=3, n_pages=14,
                        n_mem=(2,), n_win=(3,), density=Fraction(1, 2))
    prob = W.build(spec)
    fl = [int(x) for x in prob.frame_idx]
    mem, win, cur = fl[:2], fl[2:5], fl[5:]
    unused = [pg for pg in range(spec.n_pages) if pg not in fl][:4]
    z2 = torch.randn(4096).cuda()
    z1 = z2 + 0.1                                        # D = 0.01; kappa = 0.01, L_max = 6 -> 6 * 0.01 / 0.02 = 3
    ema = torch.zeros(2, dtype=torch.float32, device="cuda")
    out = torch.full((16,), -7, dtype=torch.int32, device="cuda")
    res = torch.zeros(24, dtype=torch.uint8, device="cuda")
    ws = torch.empty(li.lib().li_policy_workspace_bytes(), dtype=torch.uint8, device="cuda")
    li.li_context_policy(z1, z2, ema, 1.0, 0.0100001, 6, _dev([0.9], torch.float32), 0.45, _dev(mem, torch.int32),
                         _dev(unused + win, torch.int32), _dev(cur, torch.int32), out, res, ws, round_nearest=True)
    r = li.policy_result(res)
    assert r.L_t == 3 and r.keep_memory == 1 and r.n_frames == len(fl)
    np.testing.assert_array_equal(out[:r.n_frames].cpu().numpy(), prob.frame_idx)
    ctx_ref, buf_ref = P.run_gpu(prob)
    ctx = li.Context(prob.q.cuda(), prob.k_cache.cuda(), prob.v_cache.cuda(), out[:r.n_frames], [0, r.n_frames],
                     spec.n_cur_frames, spec.block)
    buf = li.Buffers(ctx, prob.kmax)
    li.forward(ctx, prob.top_k, buf)
    torch.cuda.synchronize()
    assert torch.equal(buf.sel_idx, buf_ref.sel_idx) and torch.equal(buf.o, buf_ref.o)
