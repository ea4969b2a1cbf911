"""Pins for the oracle's frame times and pointing jitter ("the line of the trajectory
(including the pointing jitter)", L116 "the time-jump that occurs when TESS is transmitting frames"):
    c_t = (x, y) + v (tau_t - t0) + a (tau_t - t0)^2 + j_t.
Each check compares the oracle with something other than itself.  No GPU needed."""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle


def _fr(v) -> Fraction:
    return Fraction(float(np.float32(v)))


def _shift_phase(v, a, tau, t0, j):
    dt = _fr(tau) - _fr(t0)
    d = _fr(v) * dt + _fr(a) * dt * dt + _fr(j)
    s = math.floor(d + Fraction(1, 2))
    return s, float(d - s)


def brute_point(frames, sigma_t, traj, prf_sigma, t0, x, y, times, jitter):
    """Exact-rational displacements, math.exp per tap, math.fsum -- shares nothing with the oracle."""
    T, H, W = frames.shape
    two_s2 = 2.0 * float(np.float32(prf_sigma)) ** 2
    n_terms, d_terms = [], []
    for t in range(T):
        sx, phx = _shift_phase(traj[0], traj[2], times[t], t0, jitter[t][0])
        sy, phy = _shift_phase(traj[1], traj[3], times[t], t0, jitter[t][1])
        q = 1.0 / float(sigma_t[t]) ** 2
        for i in (-2, -1, 0, 1, 2):
            for j in (2, 1, 0, -1, -2):
                px, py = x + sx + i, y + sy + j
                if 0 <= px < W and 0 <= py < H:
                    g = math.exp(-((i - phx) ** 2 + (j - phy) ** 2) / two_s2)
                    n_terms.append(g * float(frames[t, py, px]) * q)
                    d_terms.append(g * g * q)
    N, D = math.fsum(n_terms), math.fsum(d_terms)
    return (N / math.sqrt(D) if D > 0 else 0.0), N, D


def _case(seed, T=6, H=12, W=14):
    rng = np.random.default_rng(seed)
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    sig = rng.uniform(0.8, 1.2, T).astype(np.float32)
    # a gap in the middle of the sequence, quarter-frame time stamps (exact in float32)
    times = (np.arange(T) + np.where(np.arange(T) >= T // 2, 7.25, 0.0)).astype(np.float32)
    jitter = (rng.integers(-6, 7, size=(T, 2)) / 8.0).astype(np.float32)      # eighths of a pixel
    return f, sig, times, jitter


@pytest.mark.parametrize("traj", [(0.3, -0.2, 0.0, 0.0), (0.11, 0.07, 0.003, -0.002), (0.0, 0.0, 0.0, 0.0)])
def test_point_matches_exact_rational_brute_force(traj):
    f, sig, times, jitter = _case(1)
    tr = np.array(traj, np.float32)
    for (x, y) in [(0, 0), (5, 6), (13, 11), (2, 9)]:
        s, N, D = oracle.point(f, sig, tr, 1.0, 3.5, x, y, times=times, jitter=jitter)
        bs, bN, bD = brute_point(f, sig, tr, 1.0, 3.5, x, y, times, jitter)
        assert N == pytest.approx(bN, rel=1e-12, abs=1e-13)
        assert D == pytest.approx(bD, rel=1e-12) and s == pytest.approx(bs, rel=1e-12, abs=1e-13)


def test_map_matches_point_and_defaults_are_frame_index_and_zero_jitter():
    f, sig, times, jitter = _case(2)
    trs = np.array([[0.3, -0.2, 0, 0], [0.1, 0.25, 0.01, 0]], np.float32)
    m = oracle.snr_map(f, sig, trs, 1.0, 2.0, times=times, jitter=jitter)
    for k in range(2):
        for y in range(0, 12, 3):
            for x in range(0, 14, 3):
                assert m[k, y, x] == pytest.approx(
                    oracle.point(f, sig, trs[k], 1.0, 2.0, x, y, times=times, jitter=jitter)[0], rel=1e-12, abs=1e-13)
    T = f.shape[0]
    base = oracle.snr_map(f, sig, trs, 1.0, 2.0)
    same = oracle.snr_map(f, sig, trs, 1.0, 2.0, times=np.arange(T, dtype=np.float32),
                          jitter=np.zeros((T, 2), np.float32))
    assert np.array_equal(base, same)
    assert not np.array_equal(base, m)


def test_time_rescaling_is_a_velocity_rescaling():
    """tau -> 2 tau, t0 -> 2 t0, v -> v/2, a -> a/4 leaves every displacement unchanged (powers of two:
    exact in floating point), so the maps are bitwise equal."""
    f, sig, _, _ = _case(3)
    T = f.shape[0]
    trs = np.array([[0.3, -0.2, 0.004, 0], [0.1, 0.25, 0, -0.008]], np.float32)
    a = oracle.snr_map(f, sig, trs, 1.0, 2.5)
    trs2 = trs * np.array([0.5, 0.5, 0.25, 0.25], np.float32)
    b = oracle.snr_map(f, sig, trs2, 1.0, 5.0, times=2.0 * np.arange(T, dtype=np.float32))
    assert np.array_equal(a, b)


def test_integer_jitter_is_a_shift_of_the_frames():
    """With whole-pixel jitter j_t the numerator equals that of the un-jittered search on frames whose
    content is moved by -j_t (zero fill), wherever no tap leaves the frame."""
    rng = np.random.default_rng(4)
    T, H, W = 5, 30, 32
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    sig = rng.uniform(0.8, 1.2, T).astype(np.float32)
    jit = rng.integers(-3, 4, size=(T, 2)).astype(np.float32)
    moved = np.zeros_like(f)
    for t in range(T):
        jx, jy = int(jit[t, 0]), int(jit[t, 1])
        src = f[t, max(0, jy):H + min(0, jy), max(0, jx):W + min(0, jx)]
        moved[t, max(0, -jy):H + min(0, -jy), max(0, -jx):W + min(0, -jx)] = src
    trs = np.array([[0.3, -0.2, 0, 0], [0.0, 0.4, 0, 0.01]], np.float32)
    _, Nj, Dj = oracle.snr_map(f, sig, trs, 1.0, 2.0, jitter=jit, return_ND=True)
    _, N0, D0 = oracle.snr_map(moved, sig, trs, 1.0, 2.0, return_ND=True)
    core = (slice(None), slice(8, H - 8), slice(8, W - 8))
    assert np.allclose(Nj[core], N0[core], rtol=0, atol=1e-12)
    assert np.allclose(Dj[core], D0[core], rtol=1e-14)


@pytest.mark.parametrize("traj", [(0.31, -0.17, 0.0, 0.0), (0.05, 0.12, 0.004, 0.003)])
def test_closed_form_injected_source_with_times_and_jitter(traj):
    """Noiseless stack with one source rendered on the same track: N/D = A and SNR = A sqrt(D)."""
    _, sig, times, jitter = _case(5, T=8, H=40, W=40)
    tr = np.array(traj, np.float32)
    frames = np.zeros((8, 40, 40), np.float32)
    oracle.inject(frames, tr[None], [20], [19], [2.5], 1.0, 4.0, times=times, jitter=jitter)
    # the renderer itself against a direct evaluation of A g at one tap of one frame
    t = 5
    sx, phx = _shift_phase(tr[0], tr[2], times[t], 4.0, jitter[t][0])
    sy, phy = _shift_phase(tr[1], tr[3], times[t], 4.0, jitter[t][1])
    assert frames[t, 19 + sy + 1, 20 + sx - 1] == pytest.approx(
        2.5 * math.exp(-((-1 - phx) ** 2 + (1 - phy) ** 2) / 2.0), rel=1e-6)
    s, N, D = oracle.point(frames, sig, tr, 1.0, 4.0, 20, 19, times=times, jitter=jitter)
    assert N / D == pytest.approx(2.5, rel=1e-6)
    assert s == pytest.approx(2.5 * math.sqrt(D), rel=1e-6)
    # without the jitter the filter is mismatched: strictly less SNR
    assert oracle.point(frames, sig, tr, 1.0, 4.0, 20, 19, times=times)[0] < s
