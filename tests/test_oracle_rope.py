"""Pins of oracle.rope (second half; reading N1-4) against what the
mathematics of a rotation fixes -- none of them restates the oracle's formula:
position 0 is the identity; every (i, i + D/2) pair keeps its norm; rotating twice adds the
positions; <R_m q, R_n k> depends on m - n only (the property the embedding exists for); the first
pair turns by exactly `position` radians and the last by position * theta^(-(D-2)/D); a transposed
pairing (i, i+1) or a flipped sign fails the hand-computed quarter turn."""
import numpy as np

import oracle


def _x(T, H, D, seed):
    return np.random.default_rng(seed).standard_normal((T, H, D))


def test_position_zero_is_identity():
    x = _x(5, 3, 64, 0)
    assert np.array_equal(oracle.rope(x, np.zeros(5, np.int32), 1e6), x)


def test_pair_norms_are_kept():
    x = _x(9, 2, 128, 1)
    y = oracle.rope(x, np.arange(9) * 977, 1e4)
    n = lambda z: z[..., :64] ** 2 + z[..., 64:] ** 2
    assert np.allclose(n(y), n(x), rtol=1e-12, atol=0)


def test_rotations_add():
    x = _x(4, 2, 64, 2)
    a, b = np.array([3, 100, 4096, 31000]), np.array([7, 23, 5000, 14000])
    twice = oracle.rope(oracle.rope(x, a, 1e6), b, 1e6)
    assert np.allclose(twice, oracle.rope(x, a + b, 1e6), rtol=0, atol=1e-9)


def test_scores_depend_on_relative_position_only():
    D = 128
    q, k = _x(1, 1, D, 3), _x(1, 1, D, 4)
    for m, n in [(10, 3), (40000, 39993), (1234, 1227)]:
        s1 = np.sum(oracle.rope(q, [m], 1e6) * oracle.rope(k, [n], 1e6))
        s0 = np.sum(oracle.rope(q, [m - n], 1e6) * k)
        assert abs(s1 - s0) < 1e-8


def test_first_and_last_frequency_by_hand():
    D, theta, p = 64, 1e4, 3
    x = np.zeros((1, 1, D))
    x[0, 0, 0] = 1.0          # pair (0, 32): turns by p radians
    x[0, 0, 31] = 2.0         # pair (31, 63): turns by p * theta^(-62/64)
    y = oracle.rope(x, [p], theta)[0, 0]
    assert abs(y[0] - np.cos(3.0)) < 1e-15 and abs(y[32] - np.sin(3.0)) < 1e-15
    a = 3.0 * theta ** (-62.0 / 64.0)
    assert abs(y[31] - 2 * np.cos(a)) < 1e-15 and abs(y[63] - 2 * np.sin(a)) < 1e-15
    assert np.count_nonzero(y) == 4


def test_quarter_turn_sign_and_pairing():
    # theta = 1 makes every frequency 1: position pi/2 is not an integer, so use the w_0 = 1 pair
    # with an angle whose sine and cosine are known: p = 11, 11 rad = 2 pi + 4.7168 -> (cos, sin) =
    # (0.0044257, -0.9999902); x = e_0 must land on (cos, sin) in slots (0, D/2), not (0, 1)
    D = 64
    x = np.zeros((1, 1, D))
    x[0, 0, 0] = 1.0
    y = oracle.rope(x, [11], 1e6)[0, 0]
    assert abs(y[0] - 0.004425697988050785) < 1e-12 and abs(y[D // 2] + 0.9999902065507035) < 1e-12
    assert y[1] == 0.0
