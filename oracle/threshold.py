"""Oracle for F1 — thresholding the demagnetisation tensor (§4.3.1).

TEST INFRASTRUCTURE ONLY (same rules as mt_oracle.py): plain numpy, the definition written out.

PAPER.md:239: "A threshold is chosen and the values which in absolute value is smaller than the
threshold is set to zero.  For example for a threshold of 20% the absolute smallest fifth of the
elements larger than zero in the tensor is truncated to zero."

Reading (Q20): "the tensor" is the dense 3N x 3N matrix of Eq. 17, so an
off-diagonal component N^{ab} = N^{ba} (stored once in the six-plane layout) counts twice among "the
elements"; exact zeros are not elements "larger than zero" and are never counted.  With the c
non-zero elements sorted by absolute value, a fraction X removes the first k = floor(X c) of them:
the threshold is tau = |v|_(k) (the smallest value kept) and every entry with |v| < tau becomes
zero.  Entries tied with tau are kept (the text says "smaller than the threshold").  k >= c gives
tau = +inf (everything removed); k = 0 removes nothing.
PARITY UNPINNED for the tie/multiplicity reading itself (the paper prints no number for it); the
functions are pinned to hand-computed cases in tests/test_oracle_threshold.py.
"""
from __future__ import annotations

import numpy as np

MULTIPLICITY = (1, 2, 2, 1, 2, 1)  # xx, xy, xz, yy, yz, zz in the 3N x 3N matrix


def threshold_value(N6: np.ndarray, fraction: float) -> float:
    """tau for planes N6[6][rows][n] (any float dtype; compared in that dtype) and a fraction in [0, 1]."""
    assert N6.shape[0] == 6
    parts = []
    for c in range(6):
        a = np.abs(N6[c]).ravel()
        a = a[a > 0]
        parts.extend([a] * MULTIPLICITY[c])
    allv = np.sort(np.concatenate(parts))
    count = allv.size
    k = int(np.floor(fraction * count))
    if k >= count:
        return float("inf")
    return float(allv[k])


def truncate(N6: np.ndarray, tau: float) -> np.ndarray:
    """Copy of N6 with every entry of absolute value below tau set to zero."""
    out = N6.copy()
    out[np.abs(out) < tau] = 0
    return out


def kept_fraction(N6: np.ndarray, tau: float) -> float:
    """Stored entries (six-plane layout, no multiplicity) that survive tau — non-zero and not below it —
    as a fraction of all stored entries 6*rows*n: what the footprint of a sparse layout scales with."""
    a = np.abs(N6)
    return float(np.count_nonzero((a >= tau) & (a > 0))) / N6.size
