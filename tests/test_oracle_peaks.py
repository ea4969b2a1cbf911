"""Pins for the oracle's non-maximum suppression (oracle.peaks): an independent library routine on maps without
ties, a literal pixel-by-pixel loop on tiny maps with ties, hand-made examples, and the separation property."""
import numpy as np
import scipy.ndimage

import oracle


def test_distinct_values_equal_a_maximum_filter():
    rng = np.random.default_rng(0)
    z = rng.standard_normal((37, 53))
    for r in (1, 2, 5):
        ref = (z == scipy.ndimage.maximum_filter(z, size=2 * r + 1, mode="constant", cval=-np.inf)) & (z >= 0.5)
        assert np.array_equal(oracle.peaks(z, r, 0.5), ref)


def test_ties_by_literal_loop():
    rng = np.random.default_rng(1)
    z = rng.integers(0, 4, (9, 11)).astype(np.float64)            # many equal scores
    r = 2
    ref = np.zeros(z.shape, bool)
    for y in range(z.shape[0]):
        for x in range(z.shape[1]):
            ok = z[y, x] >= 1.0
            for yy in range(max(0, y - r), min(z.shape[0], y + r + 1)):
                for xx in range(max(0, x - r), min(z.shape[1], x + r + 1)):
                    if (yy, xx) == (y, x):
                        continue
                    if z[yy, xx] > z[y, x] or (z[yy, xx] == z[y, x] and (yy, xx) < (y, x)):
                        ok = False
            ref[y, x] = ok
    assert np.array_equal(oracle.peaks(z, r, 1.0), ref)


def test_hand_made_cases_and_separation():
    z = np.zeros((7, 9))
    z[3, 4] = 5.0
    z[3, 5] = 4.0                      # shoulder of the same object
    z[0, 0] = 3.0                      # a second object in the corner
    k = oracle.peaks(z, 2, 1.0)
    assert sorted(map(tuple, np.argwhere(k))) == [(0, 0), (3, 4)]
    plateau = np.zeros((5, 5))
    plateau[1:3, 1:3] = 2.0            # four equal pixels: the first in row-major order survives
    assert list(map(tuple, np.argwhere(oracle.peaks(plateau, 1, 1.0)))) == [(1, 1)]
    assert oracle.peaks(np.ones((4, 4)), 1, 2.0).sum() == 0       # nothing above the threshold
    assert oracle.peaks(np.ones((4, 4)), 0, 0.0).all()            # radius 0: every pixel above the threshold
    rng = np.random.default_rng(2)
    m = rng.standard_normal((60, 60))
    ys, xs = np.nonzero(oracle.peaks(m, 3, -np.inf))
    d = np.maximum(np.abs(ys[:, None] - ys[None, :]), np.abs(xs[:, None] - xs[None, :]))
    np.fill_diagonal(d, 99)
    assert d.min() > 3                 # no two peaks within the radius of each other
