"""Pins for the oracle's per-pixel validity weights (bright pixels are set to 0; here they
also leave the normalisation):  N = sum g F / sigma^2 with the frames F as given (F = R * valid),
D = sum g^2 valid / sigma^2.  Each check compares the oracle with something other than itself."""
import math

import numpy as np
import pytest

import oracle


def brute(frames, valid, sigma_t, traj, t0, x, y):
    """Direct double loop in Python floats, shifts by exact rounding of v*dt (no accelerations here)."""
    T, H, W = frames.shape
    N = D = 0.0
    for t in range(T):
        dt = t - t0
        dx, dy = float(np.float32(traj[0])) * dt, float(np.float32(traj[1])) * dt
        sx, sy = math.floor(dx + 0.5), math.floor(dy + 0.5)
        q = 1.0 / float(sigma_t[t]) ** 2
        for j in range(-2, 3):
            for i in range(-2, 3):
                px, py = x + sx + i, y + sy + j
                if 0 <= px < W and 0 <= py < H:
                    g = math.exp(-((i - (dx - sx)) ** 2 + (j - (dy - sy)) ** 2) / 2.0)
                    N += g * float(frames[t, py, px]) * q
                    D += g * g * float(valid[t, py, px]) * q
    return (N / math.sqrt(D) if D > 0 else 0.0), N, D


def _case(seed, T=5, H=14, W=16):
    rng = np.random.default_rng(seed)
    valid = (rng.uniform(size=(T, H, W)) > 0.3).astype(np.float32)
    frames = (rng.standard_normal((T, H, W)).astype(np.float32) * valid).astype(np.float32)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    return frames, valid, sigma


def test_point_and_map_match_brute_force_with_holes():
    f, v, sig = _case(1)
    tr = np.array([0.3, -0.45, 0, 0], np.float32)
    m, mN, mD = oracle.snr_map(f, sig, tr[None], 1.0, 2.0, valid=v, return_ND=True)
    for (x, y) in [(0, 0), (7, 6), (15, 13), (3, 11)]:
        s, N, D = oracle.point(f, sig, tr, 1.0, 2.0, x, y, valid=v)
        bs, bN, bD = brute(f, v, sig, tr, 2.0, x, y)
        assert N == pytest.approx(bN, rel=1e-12, abs=1e-13) and D == pytest.approx(bD, rel=1e-12)
        assert s == pytest.approx(bs, rel=1e-12, abs=1e-13)
        assert m[0, y, x] == pytest.approx(s, rel=1e-12, abs=1e-13)
        assert mD[0, y, x] == pytest.approx(D, rel=1e-12)


def test_all_valid_is_the_unmasked_search_and_all_masked_is_zero():
    f, v, sig = _case(2)
    trs = np.array([[0.3, -0.2, 0, 0], [0.0, 0.1, 0.01, 0]], np.float32)
    ones = np.ones_like(f)
    assert np.array_equal(oracle.snr_map(f, sig, trs, 1.0, 2.0, valid=ones), oracle.snr_map(f, sig, trs, 1.0, 2.0))
    zeros = np.zeros_like(f)
    assert np.all(oracle.snr_map(zeros, sig, trs, 1.0, 2.0, valid=zeros) == 0)       # D = 0 -> SNR = 0


def test_masked_source_keeps_n_over_d_and_loses_snr():
    """A noiseless source seen through a mask: N = A sum g^2 m / sigma^2 = A D, so N / D = A and
    SNR = A sqrt(D) with the reduced D."""
    T, H, W = 8, 30, 30
    rng = np.random.default_rng(3)
    sig = rng.uniform(0.8, 1.2, T).astype(np.float32)
    tr = np.array([0.31, -0.17, 0.003, 0], np.float32)
    frames = np.zeros((T, H, W), np.float32)
    oracle.inject(frames, tr[None], [15], [14], [1.75], 1.0, 4.0)
    valid = (rng.uniform(size=frames.shape) > 0.25).astype(np.float32)
    valid[3] = 0.0                                                                   # a whole frame lost
    masked = frames * valid
    s, N, D = oracle.point(masked, sig, tr, 1.0, 4.0, 15, 14, valid=valid)
    s0, N0, D0 = oracle.point(frames, sig, tr, 1.0, 4.0, 15, 14)
    assert N / D == pytest.approx(1.75, rel=1e-6) and s == pytest.approx(1.75 * math.sqrt(D), rel=1e-6)
    assert D < D0 and s < s0


def test_weights_scale_like_inverse_variances():
    """valid = c everywhere with frames scaled by c is the unmasked search with sigma^2 / c: SNR * sqrt(c)."""
    f, _, sig = _case(4)
    trs = np.array([[0.2, 0.25, 0, 0]], np.float32)
    base = oracle.snr_map(f, sig, trs, 1.0, 2.0)
    c = np.float32(0.25)
    got = oracle.snr_map(f * c, sig, trs, 1.0, 2.0, valid=np.full_like(f, c))
    assert np.allclose(got, base * math.sqrt(float(c)), rtol=1e-12, atol=1e-14)
