"""Pins of oracle/li_policy_oracle.py (Eq. 1-4) against what the paper and the mathematics fix:
hand-worked numbers, closed forms, limits, monotonicity, the strict inequality of Eq. 4.  CPU only."""
import numpy as np
import pytest

from oracle import li_policy_oracle as PO


def test_hand_worked_example():
    """z_{t-1} = (1,2,3,4), z_{t-2} = (1,1,1,1): squared differences 0,1,4,9 -> D = 14/4 = 3.5 (Eq. 1).
    alpha = 0.5, Dbar_{t-1} = 1.5 -> Dbar = 0.5*3.5 + 0.5*1.5 = 2.5 (Eq. 2).
    L_m = 8: kappa = 2.5 -> 8*2.5/5 = 4 exactly; kappa = 2 -> 16/4.5 = 3.55.. -> floor 3, nearest 4 (Eq. 3)."""
    D = PO.latent_mse(np.array([1., 2., 3., 4.]), np.array([1., 1., 1., 1.]))
    assert D == 3.5
    Db = PO.ema_update(D, 1.5, 0.5)
    assert Db == 2.5
    assert PO.window_length(Db, 2.5, 8) == 4 and PO.window_length(Db, 2.5, 8, "nearest") == 4
    assert PO.window_length(Db, 2.0, 8, "floor") == 3
    assert PO.window_length(Db, 2.0, 8, "nearest") == 4
    # same decisions when evaluated in the kernel's precision
    assert PO.window_length(Db, 2.0, 8, "floor", np.float32) == 3 and PO.window_length(Db, 2.0, 8, "nearest", np.float32) == 4


def test_mse_is_a_mean_over_all_dimensions_and_symmetric():
    rng = np.random.default_rng(5)
    a, b = rng.standard_normal((4, 16, 6, 7)), rng.standard_normal((4, 16, 6, 7))
    brute = 0.0
    for x, y in zip(a.ravel(), b.ravel()):
        brute += (x - y) * (x - y)
    brute /= a.size
    assert PO.latent_mse(a, b) == pytest.approx(brute, rel=1e-13)
    assert PO.latent_mse(a, b) == PO.latent_mse(b, a)
    assert PO.latent_mse(a, a) == 0.0
    # a constant offset c gives exactly c^2; scaling both by s scales D by s^2
    assert PO.latent_mse(a + 0.5, a) == pytest.approx(0.25, rel=1e-12)
    assert PO.latent_mse(3 * a, 3 * b) == pytest.approx(9 * PO.latent_mse(a, b), rel=1e-12)


def test_ema_initialisation_limits_and_fixed_point():
    assert PO.ema_update(0.7, None, 0.3) == 0.7                 # "initialized by the first valid D_t"
    assert PO.ema_update(0.7, 123.0, 1.0) == 0.7                # alpha = 1: no smoothing
    assert PO.ema_update(2.0, 2.0, 0.37) == pytest.approx(2.0)  # fixed point
    # unrolled recursion = geometric weights
    D = [0.5, 1.5, 0.25, 4.0]
    alpha = 0.25
    s = None
    for d in D:
        s = PO.ema_update(d, s, alpha)
    closed = (1 - alpha) ** 3 * D[0] + sum(alpha * (1 - alpha) ** (3 - i) * D[i] for i in range(1, 4))
    assert s == pytest.approx(closed, rel=1e-14)


@pytest.mark.parametrize("rounding", ["floor", "nearest"])
def test_window_length_limits_and_monotonicity(rounding):
    L_m, kappa = 16, 0.02
    assert PO.window_length(0.0, kappa, L_m, rounding) == L_m          # stable dynamics: whole budget
    assert PO.window_length(kappa, kappa, L_m, rounding) == L_m // 2    # Dbar = kappa: exactly half
    assert PO.window_length(1e9, kappa, L_m, rounding) == 1             # clip from below
    prev = L_m
    for Db in np.linspace(0, 1.0, 400):
        L = PO.window_length(float(Db), kappa, L_m, rounding)
        assert 1 <= L <= prev                                           # "shrinks the temporal window under large dynamics"
        prev = L
    # floor <= nearest <= floor + 1
    for Db in np.linspace(0, 0.2, 97):
        f, n = PO.window_length(float(Db), kappa, L_m, "floor"), PO.window_length(float(Db), kappa, L_m, "nearest")
        assert f <= n <= f + 1


def test_gate_is_strict_and_uses_the_maximum():
    assert PO.keep_memory([0.1, 0.7, 0.3], 0.7) is True      # max == tau: NOT "< tau" -> kept (Eq. 4 is strict)
    assert PO.keep_memory([0.1, 0.69999, 0.3], 0.7) is False
    assert PO.keep_memory([0.9, 0.0], 0.45) is True          # tau = 0.45 / 0.7 are the paper's values
    assert PO.keep_memory([], 0.45) is False


def test_frame_list_order_and_truncation():
    mem, win, cur = [40, 3], [10, 11, 12, 13, 14], [20, 21]
    np.testing.assert_array_equal(PO.reconstruct_frame_list(mem, win, cur, 2, True), [40, 3, 13, 14, 20, 21])
    np.testing.assert_array_equal(PO.reconstruct_frame_list(mem, win, cur, 2, False), [13, 14, 20, 21])
    np.testing.assert_array_equal(PO.reconstruct_frame_list(mem, win, cur, 9, False), [10, 11, 12, 13, 14, 20, 21])
    np.testing.assert_array_equal(PO.reconstruct_frame_list([], win, cur, 1, True), [14, 20, 21])
    assert PO.reconstruct_frame_list(mem, win, cur, 2, True).dtype == np.int32
    # the tiny config's list {0,3} | {6} | {7} (BASELINE.json configs[0]) is memory | window | chunk
    np.testing.assert_array_equal(PO.reconstruct_frame_list([0, 3], [5, 6], [7], 1, True), [0, 3, 6, 7])


def test_whole_policy_composes_the_steps():
    rng = np.random.default_rng(11)
    z1 = rng.standard_normal(1000)
    z2 = z1 + 0.1                                    # D = 0.01 exactly (up to rounding)
    D, Db, L, keep, fl = PO.context_policy(z1, z2, None, 0.5, 0.01, 12, [0.2, 0.5], 0.45, [7, 8], list(range(100, 112)), [1, 2])
    assert D == pytest.approx(0.01, rel=1e-9) and Db == D
    assert L in (5, 6) and keep is True            # 12 * 0.01 / 0.02 = 6 up to the rounding of D
    np.testing.assert_array_equal(fl[:2], [7, 8])
    np.testing.assert_array_equal(fl[-2:], [1, 2])
    assert len(fl) == 2 + L + 2 and fl[2] == 112 - L
