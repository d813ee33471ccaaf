"""Pins of the thresholding oracle (oracle/threshold.py): hand-computed cases."""
import numpy as np

from oracle import threshold as T


def planes(vals):
    """six 1x1 planes from six numbers"""
    return np.array(vals, dtype=np.float64).reshape(6, 1, 1)


def test_hand_case_with_multiplicity():
    # 3x3 block [[5, 1, 2], [1, 6, 3], [2, 3, 7]]: elements sorted by |.|: 1, 1, 2, 2, 3, 3, 5, 6, 7 (c = 9)
    N = planes([5, 1, -2, 6, 3, -7])
    assert T.threshold_value(N, 0.0) == 1.0          # k = 0: nothing removed
    assert T.threshold_value(N, 0.2) == 1.0          # k = 1: the tie with the removed element is kept
    assert T.threshold_value(N, 2 / 9) == 2.0        # k = 2: both copies of xy go
    assert T.threshold_value(N, 0.5) == 3.0          # k = 4
    assert T.threshold_value(N, 0.7) == 5.0          # k = 6
    assert T.threshold_value(N, 1.0) == float("inf")
    out = T.truncate(N, 3.0)
    assert out.ravel().tolist() == [5, 0, 0, 6, 3, -7]
    assert T.truncate(N, float("inf")).any() == False  # noqa: E712


def test_zeros_are_not_elements():
    # PAPER.md:239 "of the elements larger than zero": zeros neither count nor move the threshold
    N = np.zeros((6, 2, 2))
    N[0] = [[4, 0], [0, 8]]
    N[3] = [[0, 2], [6, 0]]
    # non-zero elements: 2, 4, 6, 8
    assert T.threshold_value(N, 0.25) == 4.0
    assert T.threshold_value(N, 0.5) == 6.0
    assert T.kept_fraction(N, 6.0) == 2 / 24


def test_distinct_values_remove_exactly_k():
    rng = np.random.default_rng(0)
    N = rng.normal(size=(6, 5, 7))
    mult = np.array(T.MULTIPLICITY).reshape(6, 1, 1) * np.ones_like(N)
    for X in (0.1, 0.35, 0.8):
        tau = T.threshold_value(N, X)
        removed = mult[np.abs(N) < tau].sum()
        k = np.floor(X * mult.sum())
        assert k - 1 <= removed <= k  # an off-diagonal pair straddling k is kept whole or removed whole
        kept = T.truncate(N, tau)
        assert np.array_equal(kept[np.abs(N) >= tau], N[np.abs(N) >= tau])


def test_float32_planes_compare_in_float32():
    N = np.array([1.0, 1.0 + 2**-23, 3, 4, 5, 6], dtype=np.float32).reshape(6, 1, 1)
    assert T.threshold_value(N, 0.12) == float(np.float32(1.0 + 2**-23))
