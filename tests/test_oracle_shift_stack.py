"""Pins for the oracle's shift-stack mode (after Rice & Laughlin 2020: "a single non-zero
value, set to 1, for each time-slice"): the filter is 1 at the rounded position of the track and 0 elsewhere,
N = sum_t R_t(round(c_t)) / sigma_t^2, D = sum_t [in frame] / sigma_t^2."""
import math

import numpy as np
import pytest

import oracle


def test_shift_stack_is_a_sum_of_shifted_frames():
    rng = np.random.default_rng(1)
    T, H, W = 7, 20, 24
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    sig = rng.uniform(0.8, 1.2, T).astype(np.float32)
    trs = np.array([[0.6, -0.4, 0, 0], [0.25, 0.0, 0, 0.05]], np.float32)
    t0 = 3.0
    m, N, D = oracle.snr_map(f, sig, trs, 1.0, t0, shift_stack=True, return_ND=True)
    for k, tr in enumerate(trs):
        n = np.zeros((H, W)); d = np.zeros((H, W))
        for t in range(T):
            dt = t - t0
            sx = math.floor(float(tr[0]) * dt + float(tr[2]) * dt * dt + 0.5)
            sy = math.floor(float(tr[1]) * dt + float(tr[3]) * dt * dt + 0.5)
            q = 1.0 / float(sig[t]) ** 2
            for y in range(H):
                for x in range(W):
                    if 0 <= x + sx < W and 0 <= y + sy < H:
                        n[y, x] += float(f[t, y + sy, x + sx]) * q
                        d[y, x] += q
        assert np.allclose(N[k], n, rtol=0, atol=1e-12) and np.allclose(D[k], d, rtol=1e-14)
        assert np.allclose(m[k], np.where(d > 0, n / np.sqrt(np.where(d > 0, d, 1)), 0), rtol=0, atol=1e-12)
    # the point form agrees, and prf_sigma plays no role
    s1 = oracle.point(f, sig, trs[0], 1.0, t0, 5, 6, shift_stack=True)[0]
    s2 = oracle.point(f, sig, trs[0], 2.5, t0, 5, 6, shift_stack=True)[0]
    assert s1 == s2 == pytest.approx(m[0, 6, 5], abs=1e-13)


def test_matched_filter_beats_shift_stack_on_an_injected_source():
    """The paper's argument (L118): the single-pixel filter throws signal away.  For a noiseless source of
    amplitude A the matched filter has SNR = A sqrt(D) = A sqrt(sum g^2 q); the shift-stack collects only the
    peak-pixel samples, SNR = A sum(g_peak q) / sqrt(sum q).  Both closed forms are checked, and their ratio."""
    T, H, W = 40, 40, 40
    sig = np.ones(T, np.float32)
    tr = np.array([0.137, -0.081, 0, 0], np.float32)
    frames = np.zeros((T, H, W), np.float32)
    A = 2.0
    oracle.inject(frames, tr[None], [20], [20], [A], 1.0, 20.0)
    s_mf, _, D = oracle.point(frames, sig, tr, 1.0, 20.0, 20, 20)
    s_ss, N_ss, D_ss = oracle.point(frames, sig, tr, 1.0, 20.0, 20, 20, shift_stack=True)
    assert s_mf == pytest.approx(A * math.sqrt(D), rel=1e-6)
    peak = 0.0
    for t in range(T):
        dt = t - 20.0
        dx, dy = float(tr[0]) * dt, float(tr[1]) * dt
        phx, phy = dx - math.floor(dx + 0.5), dy - math.floor(dy + 0.5)
        peak += math.exp(-(phx * phx + phy * phy) / 2.0)
    assert D_ss == pytest.approx(T) and N_ss == pytest.approx(A * peak, rel=1e-6)
    assert s_ss == pytest.approx(A * peak / math.sqrt(T), rel=1e-6)
    # Gaussian PRF of width 1 px: sum g^2 ~ pi per frame, peak sample ~ 0.92 on average -> ratio ~ 1.9
    assert 1.7 < s_mf / s_ss < 2.1
