"""Philox4x32-10 of the oracle against the published known-answer vectors (CPU only)."""
import os

import numpy as np

from oracle import sw_oracle as so
from stats import golden_rows

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers():
    rows = golden_rows(GOLD)
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert so.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_philox_words_are_uniform_and_distinct_per_domain():
    """Coarse sanity of the keying: different sites / steps / seeds / domains give different words
    and the top bits are balanced (a stuck counter or key word would fail this)."""
    w = np.array([so.philox4x32_10([i, t, 0, 0], [1, 0]) for i in range(64) for t in range(64)], dtype=np.uint64)
    assert len(np.unique(w[:, 0])) == len(w)
    frac = (w >> 31).mean(axis=0)
    assert np.all(np.abs(frac - 0.5) < 4 * 0.5 / np.sqrt(len(w)))
    base = so.philox4x32_10([5, 0, 0, 0], [1, 0])
    assert base != so.philox4x32_10([5, 0, 0, 0], [2, 0])
    assert base != so.philox4x32_10([5, 0, 0, 0], [1, 1])
    assert base != so.philox4x32_10([5, 0, 1, 0], [1, 0])
    assert base != so.philox4x32_10([5, 0, 0, 2], [1, 0])
