"""Pins for the CPU oracle (oracle/tno_oracle.c): every check here compares the oracle with
something other than itself -- a closed form, an invariant, a library routine on a special
case, exact-rational brute force, or hand-listed expectations.  No GPU needed.

Numbering follows BASELINE.json:north_star checks (1)-(5) and SURVEY.md section 8(c).
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.ndimage

import oracle
import tno_synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------------------------------------
# An independent, deliberately different evaluation of the definition: exact rational
# displacements (fractions.Fraction), math.exp per tap, math.fsum accumulation, taps visited
# column-major.  Shares nothing with the oracle's C code.
# ---------------------------------------------------------------------------------------------
def _frac(v) -> Fraction:
    return Fraction(float(np.float32(v)))


def _shift_phase(v, a, t, t0):
    dt = Fraction(t) - _frac(t0)
    d = _frac(v) * dt + _frac(a) * dt * dt
    s = math.floor(d + Fraction(1, 2))        # ties go up
    return s, float(d - s)


def brute_point(frames, sigma_t, traj, prf_sigma, t0, x, y):
    T, H, W = frames.shape
    two_s2 = 2.0 * float(np.float32(prf_sigma)) ** 2
    n_terms, d_terms = [], []
    for t in range(T):
        sx, phx = _shift_phase(traj[0], traj[2], t, t0)
        sy, phy = _shift_phase(traj[1], traj[3], t, t0)
        q = 1.0 / float(sigma_t[t]) ** 2
        for i in (-2, -1, 0, 1, 2):
            for j in (2, 1, 0, -1, -2):
                px, py = x + sx + i, y + sy + j
                if not (0 <= px < W and 0 <= py < H):
                    continue
                g = math.exp(-((i - phx) ** 2 + (j - phy) ** 2) / two_s2)
                n_terms.append(g * float(frames[t, py, px]) * q)
                d_terms.append(g * g * q)
    N, D = math.fsum(n_terms), math.fsum(d_terms)
    return (N / math.sqrt(D) if D > 0 else 0.0), N, D


def render_source(frames, traj, x, y, amp, prf_sigma, t0):
    """Test-local renderer (independent of oracle.inject): add amp * g on the 25 taps."""
    T, H, W = frames.shape
    two_s2 = 2.0 * float(np.float32(prf_sigma)) ** 2
    for t in range(T):
        sx, phx = _shift_phase(traj[0], traj[2], t, t0)
        sy, phy = _shift_phase(traj[1], traj[3], t, t0)
        for j in range(-2, 3):
            for i in range(-2, 3):
                px, py = x + sx + i, y + sy + j
                if 0 <= px < W and 0 <= py < H:
                    g = math.exp(-((i - phx) ** 2 + (j - phy) ** 2) / two_s2)
                    frames[t, py, px] = np.float32(float(frames[t, py, px]) + float(amp) * g)


def _rand_stack(rng, T, H, W):
    return rng.standard_normal((T, H, W)).astype(np.float32)


# ------------------------------------------------------------------ (5) brute force, tiny stacks
@pytest.mark.parametrize("traj,t0", [
    ((0.3, -0.2, 0.0, 0.0), 0.0),
    ((-0.45, 0.7, 0.0, 0.0), 2.0),
    ((0.13, 0.29, 0.02, -0.03), 1.0),
    ((1.0, -2.0, 0.0, 0.0), 1.0),
    ((0.0, 0.0, 0.0, 0.0), 0.0),
])
def test_point_matches_exact_rational_brute_force(traj, t0):
    rng = np.random.default_rng(11)
    T, H, W = 4, 7, 8
    frames = _rand_stack(rng, T, H, W)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.asarray(traj, dtype=np.float32)
    for y in range(H):
        for x in range(W):
            s, N, D = oracle.point(frames, sigma, traj, 1.1, t0, x, y)
            bs, bN, bD = brute_point(frames, sigma, traj, 1.1, t0, x, y)
            assert N == pytest.approx(bN, rel=1e-12, abs=1e-13)
            assert D == pytest.approx(bD, rel=1e-12)
            assert s == pytest.approx(bs, rel=1e-12, abs=1e-13)


def test_map_matches_point_everywhere_small():
    rng = np.random.default_rng(5)
    T, H, W = 6, 9, 11
    frames = _rand_stack(rng, T, H, W)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    trajs = np.array([[0.4, -0.3, 0.0, 0.0], [-0.9, 0.2, 0.05, 0.0], [0.0, 1.0, 0.0, -0.04]],
                     dtype=np.float32)
    m, mN, mD = oracle.snr_map(frames, sigma, trajs, 0.9, 2.0, return_ND=True)
    for k in range(3):
        for y in range(H):
            for x in range(W):
                s, N, D = oracle.point(frames, sigma, trajs[k], 0.9, 2.0, x, y)
                assert m[k, y, x] == pytest.approx(s, rel=1e-12, abs=1e-13)
                assert mN[k, y, x] == pytest.approx(N, rel=1e-12, abs=1e-13)
                assert mD[k, y, x] == pytest.approx(D, rel=1e-12)


def test_map_region_and_window_agree_with_full():
    rng = np.random.default_rng(6)
    T, H, W = 5, 40, 48
    frames = _rand_stack(rng, T, H, W)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    trajs = np.array([[1.3, -0.8, 0.0, 0.0], [-0.5, 0.5, 0.1, 0.0]], dtype=np.float32)
    full = oracle.snr_map(frames, sigma, trajs, 1.0, 2.0)
    reg = (10, 30, 8, 25)
    part = oracle.snr_map(frames, sigma, trajs, 1.0, 2.0, region=reg)
    assert np.array_equal(part, full[:, 8:25, 10:30])
    # window: a crop with halo, evaluated against the full-frame geometry
    wx0, wy0 = 2, 1
    win = np.ascontiguousarray(frames[:, wy0:34, wx0:40])
    part2 = oracle.snr_map(win, sigma, trajs, 1.0, 2.0, region=reg, window=(wx0, wy0),
                           full_shape=(H, W))
    assert np.array_equal(part2, part)
    with pytest.raises(ValueError):     # halo too small must be reported, never silently wrong
        oracle.snr_map(np.ascontiguousarray(frames[:, 8:25, 10:30]), sigma, trajs, 1.0, 2.0,
                       region=reg, window=(10, 8), full_shape=(H, W))


# ------------------------------------------------------- (1) closed form: injected noiseless source
@pytest.mark.parametrize("traj,t0,x,y", [
    ((0.23, -0.31, 0.0, 0.0), 8.0, 20, 18),        # sub-pixel velocity
    ((0.1, 0.4, 0.004, -0.006), 8.0, 17, 22),      # with acceleration
    ((-0.37, 0.05, 0.0, 0.0), 0.0, 30, 12),        # t0 = 0
    ((0.3, 0.2, 0.0, 0.0), 8.0, 1, 2),             # start pixel next to an edge (reduced D)
    ((0.6, -0.6, 0.0, 0.0), 8.0, 35, 0),           # track leaves the frame
])
def test_closed_form_injected_source(traj, t0, x, y):
    """PAPER.md:L130 'signal injection corresponds to adding a filter times a flux'; L108 'the
    result is a direct estimate of the total flux': on a noiseless stack N/D = A and
    SNR = A sqrt(D) at the source's start pixel, for non-uniform sigma_t."""
    T, H, W = 16, 36, 40
    A = 2.75
    rng = np.random.default_rng(3)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.asarray(traj, dtype=np.float32)
    frames = np.zeros((T, H, W), dtype=np.float32)
    render_source(frames, traj, x, y, A, 1.0, t0)
    s, N, D = oracle.point(frames, sigma, traj, 1.0, t0, x, y)
    assert D > 0
    assert N / D == pytest.approx(A, rel=2e-7)            # float32 rounding of the rendered taps
    assert s == pytest.approx(A * math.sqrt(D), rel=2e-7)
    # the peak of this trajectory's map is at the source
    m = oracle.snr_map(frames, sigma, traj[None, :], 1.0, t0)
    flux = m[0]  # SNR = A_hat * sqrt(D); the exact-match pixel maximises A_hat / A = 1
    assert flux[y, x] == pytest.approx(s, rel=1e-12)


def test_interior_D_closed_form_and_golden_tap_sums():
    """Single frame, v = 0, sigma_t = 1: D = (sum_i g_i^2)^2 with g_i = exp(-i^2/(2 s^2)); for
    s = 1 that is (1 + 2/e + 2/e^4)^2.  tests/golden/prf_tap_sums.txt holds the 1-D sums quoted
    in SURVEY.md 8(c) for phase 0 and phase -0.5."""
    frames = np.ones((1, 9, 9), dtype=np.float32)
    sig = np.ones(1, dtype=np.float32)
    s, N, D = oracle.point(frames, sig, np.zeros(4, np.float32), 1.0, 0.0, 4, 4)
    sum_g2 = 1 + 2 / math.e + 2 / math.e ** 4
    sum_g = 1 + 2 * math.exp(-0.5) + 2 * math.exp(-2.0)
    assert D == pytest.approx(sum_g2 ** 2, rel=1e-14)
    assert N == pytest.approx(sum_g ** 2, rel=1e-14)
    gold = {}
    with open(os.path.join(GOLDEN, "prf_tap_sums.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                sg, ph, val = line.split()
                gold[(float(sg), float(ph))] = float(val)
    # phase -0.5 is reached with v = 0.5 at dt = 1 (d = 0.5 -> shift 1, phase -0.5): T = 2, t0 = 0
    frames2 = np.ones((2, 15, 15), dtype=np.float32)
    for (sg, ph), val in gold.items():
        if ph == 0.0:
            _, _, Dg = oracle.point(frames, sig, np.zeros(4, np.float32), sg, 0.0, 4, 4)
            assert math.sqrt(Dg) == pytest.approx(val, rel=2e-5)       # 1-D sum = sqrt of 2-D
        else:
            sig2 = np.array([1e6, 1.0], dtype=np.float32)              # frame 0 weightless
            tr = np.array([0.5, 0.5, 0, 0], dtype=np.float32)
            _, _, Dg = oracle.point(frames2, sig2, tr, sg, 0.0, 7, 7)
            assert math.sqrt(Dg) == pytest.approx(val, rel=2e-5)


# ------------------------------------------------------------------------- (2) zero in, zero out
def test_zero_frames_give_zero_map_and_empty_list():
    T, H, W = 5, 12, 13
    frames = np.zeros((T, H, W), dtype=np.float32)
    sigma = np.full(T, 1.1, dtype=np.float32)
    trajs = np.array([[0.3, 0.1, 0, 0], [2.0, -3.0, 0, 0]], dtype=np.float32)
    m = oracle.snr_map(frames, sigma, trajs, 1.0, 2.0)
    assert np.all(m == 0.0)
    c = oracle.topk(m[0], 4, 5.0, 0)
    assert np.all(c["x"] == -1) and np.all(c["y"] == -1) and np.all(np.isneginf(c["snr"]))


# ---------------------------------------------------------------------------- (3) linearity in R
def test_linearity():
    rng = np.random.default_rng(8)
    T, H, W = 7, 20, 22
    R1, R2 = _rand_stack(rng, T, H, W), _rand_stack(rng, T, H, W)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    trajs = np.array([[0.4, -0.3, 0.0, 0.0], [-0.7, 0.2, 0.02, 0.01]], dtype=np.float32)
    a, b = 2.0, -0.5                                    # exact in float32
    m1 = oracle.snr_map(R1, sigma, trajs, 1.0, 3.0)
    m2 = oracle.snr_map(R2, sigma, trajs, 1.0, 3.0)
    m12 = oracle.snr_map((a * R1 + b * R2).astype(np.float32), sigma, trajs, 1.0, 3.0)
    # a*R1+b*R2 is rounded to float32 once more: tolerance ~ 1e-7 * sqrt(D)
    assert np.max(np.abs(m12 - (a * m1 + b * m2))) < 5e-6


def test_noise_scale_invariance():
    rng = np.random.default_rng(9)
    T, H, W = 6, 16, 16
    R = _rand_stack(rng, T, H, W)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    trajs = np.array([[0.25, 0.5, 0, 0]], dtype=np.float32)
    m = oracle.snr_map(R, sigma, trajs, 1.0, 0.0)
    m4 = oracle.snr_map(R * np.float32(4), sigma * np.float32(4), trajs, 1.0, 0.0)
    assert np.max(np.abs(m - m4)) < 1e-12


# --------------------------------------------- (4) integer velocities = shifted sum of correlations
@pytest.mark.parametrize("vx,vy", [(1, 0), (0, -1), (2, 1), (-1, 3), (0, 0)])
def test_integer_velocity_reduces_to_library_correlation(vx, vy):
    rng = np.random.default_rng(21)
    T, H, W = 6, 24, 28
    t0 = 2.0
    R = _rand_stack(rng, T, H, W)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    s = 1.0
    ax = np.arange(-2, 3)
    g0 = np.exp(-(ax[None, :] ** 2 + ax[:, None] ** 2) / (2 * s * s))      # [j, i], phase 0
    P = 3 * max(abs(vx), abs(vy), 1) + 4
    N = np.zeros((H, W))
    D = np.zeros((H, W))
    for t in range(T):
        q = 1.0 / float(sigma[t]) ** 2
        pad = np.zeros((H + 2 * P, W + 2 * P))
        pad[P:P + H, P:P + W] = R[t]
        ones = np.zeros_like(pad)
        ones[P:P + H, P:P + W] = 1.0
        c = scipy.ndimage.correlate(pad, g0, mode="constant", cval=0.0)
        d = scipy.ndimage.correlate(ones, g0 * g0, mode="constant", cval=0.0)
        sx, sy = vx * (t - int(t0)), vy * (t - int(t0))
        N += q * c[P + sy:P + sy + H, P + sx:P + sx + W]
        D += q * d[P + sy:P + sy + H, P + sx:P + sx + W]
    expect = np.where(D > 0, N / np.sqrt(np.where(D > 0, D, 1.0)), 0.0)
    m, mN, mD = oracle.snr_map(R, sigma, np.array([[vx, vy, 0, 0]], dtype=np.float32), s, t0,
                               return_ND=True)
    assert np.max(np.abs(mD[0] - D)) < 1e-12
    assert np.max(np.abs(mN[0] - N)) < 1e-12
    assert np.max(np.abs(m[0] - expect)) < 1e-12


# --------------------------------------------------------------------------------- tie rule (c1, c3)
def test_ties_round_up_hand_listed():
    """v = -0.5f, t0 = 0: at t = 5 the displacement is exactly -2.5 -> shift -2, phase -0.5
    (C round() would give -3).  An impulse in frame 5 only, at x_p: the start pixels that see it
    are x + (-2) + i = x_p, i in -2..2, i.e. x in [x_p, x_p + 4]; with half-away-from-zero
    rounding it would be [x_p + 1, x_p + 5].  Likewise v = +0.5f: d = 2.5 -> shift 3."""
    T, H, W = 6, 9, 30
    sigma = np.ones(T, dtype=np.float32)
    xp, yp = 15, 4
    frames = np.zeros((T, H, W), dtype=np.float32)
    frames[5, yp, xp] = 1.0
    for v, lo in ((-0.5, xp), (0.5, xp - 5)):
        m, mN, _ = oracle.snr_map(frames, sigma, np.array([[v, 0, 0, 0]], np.float32), 1.0, 0.0,
                                  return_ND=True)
        hit = np.nonzero(mN[0, yp] != 0.0)[0]
        assert hit.tolist() == list(range(lo, lo + 5)), (v, hit)
        # weights along x are g(i + 0.5) for i = -2..2 read right-to-left
        w = [math.exp(-((i + 0.5) ** 2) / 2.0) for i in (2, 1, 0, -1, -2)]
        assert mN[0, yp, lo:lo + 5] == pytest.approx(w, rel=1e-14)
    # quarter-pixel velocity: d = 0.25 * 2 = 0.5 -> shift 1; d = 0.25 * 6 = 1.5 -> shift 2
    frames[:] = 0
    frames[2, yp, xp] = 1.0
    _, mN, _ = oracle.snr_map(frames[:3], sigma[:3], np.array([[0.25, 0, 0, 0]], np.float32),
                              1.0, 0.0, return_ND=True)
    assert np.nonzero(mN[0, yp] != 0.0)[0].tolist() == list(range(xp - 3, xp + 2))


def test_config1_near_ties_resolved_like_exact_arithmetic():
    """0.1f * 5 = 0.5000000074505806 in exact arithmetic -> shift 1."""
    s, ph = _shift_phase(np.float32(0.1), 0.0, 5, 0.0)
    assert s == 1 and ph == pytest.approx(-0.4999999925, abs=1e-9)
    frames = np.zeros((6, 5, 20), dtype=np.float32)
    frames[5, 2, 10] = 1.0
    _, mN, _ = oracle.snr_map(frames, np.ones(6, np.float32),
                              np.array([[0.1, 0, 0, 0], [-0.1, 0, 0, 0]], np.float32), 1.0, 0.0,
                              return_ND=True)
    assert np.nonzero(mN[0, 2])[0].tolist() == list(range(7, 12))      # shift +1
    assert np.nonzero(mN[1, 2])[0].tolist() == list(range(9, 14))      # shift -1


# --------------------------------------------------------------------------------- borders (c8)
def test_corner_closed_form_all_ones():
    """All-ones frames, sigma_t = 1, v = 0: at (0, 0) only taps i, j >= 0 survive."""
    T = 7
    frames = np.ones((T, 10, 10), dtype=np.float32)
    sig = np.ones(T, dtype=np.float32)
    g = [math.exp(-i * i / 2.0) for i in (0, 1, 2)]
    sg, sg2 = sum(g), sum(v * v for v in g)
    expect = T * sg ** 2 / math.sqrt(T * sg2 ** 2)
    s, N, D = oracle.point(frames, sig, np.zeros(4, np.float32), 1.0, 3.0, 0, 0)
    assert s == pytest.approx(expect, rel=1e-14)
    # edge (not corner): x interior, y = 0
    full = 1 + 2 * g[1] + 2 * g[2]
    full2 = 1 + 2 * g[1] ** 2 + 2 * g[2] ** 2
    s2, _, _ = oracle.point(frames, sig, np.zeros(4, np.float32), 1.0, 3.0, 5, 0)
    assert s2 == pytest.approx(T * sg * full / math.sqrt(T * sg2 * full2), rel=1e-14)


def test_all_taps_off_frame_gives_zero():
    frames = np.ones((3, 6, 6), dtype=np.float32)
    sig = np.ones(3, dtype=np.float32)
    # t0 = -20, v = 1: displacement >= 20 px in every frame -> every tap off frame
    s, N, D = oracle.point(frames, sig, np.array([1, 0, 0, 0], np.float32), 1.0, -20.0, 2, 2)
    assert (s, N, D) == (0.0, 0.0, 0.0)


def test_mirror_symmetry():
    rng = np.random.default_rng(12)
    T, H, W = 8, 18, 21
    R = _rand_stack(rng, T, H, W)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    tr = np.array([[0.37, -0.21, 0.013, 0.004]], dtype=np.float32)      # no exact ties
    trm = tr * np.array([-1, 1, -1, 1], dtype=np.float32)
    m = oracle.snr_map(R, sigma, tr, 1.0, 4.0)
    mm = oracle.snr_map(np.ascontiguousarray(R[:, :, ::-1]), sigma, trm, 1.0, 4.0)
    assert np.max(np.abs(mm[0, :, ::-1] - m[0])) < 1e-12


# ----------------------------------------------------------- noise weighting: SNR ~ N(0,1) on noise
def test_pure_noise_map_is_unit_normal_including_edges():
    rng = np.random.default_rng(2024)
    T, H, W = 24, 96, 96
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    R = (rng.standard_normal((T, H, W)) * sigma[:, None, None]).astype(np.float32)
    trajs = np.array([[0.3, -0.2, 0, 0], [-0.45, 0.1, 0.01, 0], [0, 0, 0, 0]], dtype=np.float32)
    m = oracle.snr_map(R, sigma, trajs, 1.0, 12.0)
    # neighbouring pixels share taps: ~ (H*W)/12 effective samples per map
    for k in range(3):
        assert abs(m[k].mean()) < 0.06
        assert abs(m[k].std() - 1.0) < 0.05
        edge = np.concatenate([m[k][:2].ravel(), m[k][-2:].ravel(),
                               m[k][:, :2].ravel(), m[k][:, -2:].ravel()])
        assert abs(edge.std() - 1.0) < 0.12


# ----------------------------------------------------------------------------------- injection
def test_inject_matches_independent_renderer():
    T, H, W = 10, 30, 32
    trajs = np.array([[0.31, -0.17, 0, 0], [-0.6, 0.4, 0.01, -0.02], [0.2, 0.2, 0, 0]],
                     dtype=np.float32)
    xs, ys = np.array([10, 20, 1], np.int32), np.array([12, 8, 28], np.int32)
    amps = np.array([3.0, 1.25, 0.7], np.float32)
    rng = np.random.default_rng(4)
    base = _rand_stack(rng, T, H, W)
    a = base.copy()
    oracle.inject(a, trajs, xs, ys, amps, 1.2, 5.0)
    b = base.copy()
    for m in range(3):
        render_source(b, trajs[m], int(xs[m]), int(ys[m]), float(amps[m]), 1.2, 5.0)
    assert np.array_equal(a, b)
    assert np.count_nonzero(a != base) > 25 * T


# --------------------------------------------------------------------------------------- top-K
def _py_topk(m, ktop, thr):
    H, W = m.shape
    c = [(-m[y, x], y, x) for y in range(H) for x in range(W) if m[y, x] >= thr]
    c.sort()
    return [(-v, x, y) for v, y, x in c[:ktop]]


def test_topk_against_python_sort_and_padding():
    rng = np.random.default_rng(17)
    m = rng.standard_normal((23, 19)) * 3
    for ktop, thr in ((5, 2.0), (40, 5.0), (3, -np.inf), (4, 100.0)):
        c = oracle.topk(m, ktop, thr, 7)
        ref = _py_topk(m, ktop, thr)
        n = len(ref)
        assert [(float(r["snr"]), int(r["x"]), int(r["y"])) for r in c[:n]] == ref
        assert np.all(c["k"] == 7)
        assert np.all(c["x"][n:] == -1) and np.all(np.isneginf(c["snr"][n:]))


def test_topk_exact_ties_order_by_y_then_x_and_threshold_is_inclusive():
    m = np.zeros((6, 6))
    m[4, 1] = m[1, 4] = m[1, 2] = m[3, 3] = 7.0
    m[0, 0] = 5.0                                   # == threshold: included
    m[5, 5] = np.nextafter(5.0, 0.0)                # just below: excluded
    c = oracle.topk(m, 8, 5.0, 0)
    got = [(int(r["y"]), int(r["x"])) for r in c if r["x"] >= 0]
    assert got == [(1, 2), (1, 4), (3, 3), (4, 1), (0, 0)]
    # two identical, well separated impulses produce exact ties in the oracle's own map
    R = np.zeros((4, 12, 24), dtype=np.float32)
    R[:, 5, 6] = 2.0
    R[:, 5, 17] = 2.0
    mm = oracle.snr_map(R, np.ones(4, np.float32), np.zeros((1, 4), np.float32), 1.0, 0.0)[0]
    assert np.array_equal(mm[:, 1:12], mm[:, 12:23])
    c = oracle.topk(mm, 12, 0.5, 0)
    assert c["snr"][0] == c["snr"][1] and (c["x"][0], c["x"][1]) == (6, 17)
    # the next ring is a 4-way tie within a row and across the two blobs
    assert len(set(c["snr"][2:6].tolist())) == 1
    assert [(int(r["snr"] * 0 + r["y"]), int(r["x"])) for r in c[2:6]] == \
        sorted((int(r["y"]), int(r["x"])) for r in c[2:6])
    assert [(float(r["snr"]), int(r["x"]), int(r["y"])) for r in c] == _py_topk(mm, 12, 0.5)


# ------------------------------------------------------------- generated regression fixture
def test_config1_golden_regression():
    """tests/golden/cfg1_oracle.txt is written by tests/golden/make_golden.py, which calls only
    oracle/ and tno_synth/: guards the oracle and the generator against accidental change."""
    p = tno_synth.make_params(tno_synth.CONFIGS[1])
    f = tno_synth.stack_numpy(p)
    oracle.inject(f, p.traj[p.src_k], p.src_x, p.src_y, p.src_amp, p.cfg.prf_sigma, p.cfg.t0)
    with open(os.path.join(GOLDEN, "cfg1_oracle.txt")) as fh:
        rows = [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]
    assert len(rows) >= 9
    for k, x, y, val in rows:
        s, _, _ = oracle.point(f, p.sigma_t, p.traj[int(k)], p.cfg.prf_sigma, p.cfg.t0,
                               int(x), int(y))
        assert s == pytest.approx(float(val), rel=1e-12, abs=1e-12)


# ---------------------------------------------------------------------------------------------
# Interpreting scores (section 3.3): max over the filter bank (L112), scores in units of
# the standard deviation of the scores in the box centred on a pixel (L124).
def test_best_is_max_and_first_argmax():
    rng = np.random.default_rng(5)
    s = rng.integers(-3, 4, size=(7, 9, 11)).astype(np.float32)      # many exact ties
    m, a = oracle.best(s)
    assert np.array_equal(m, s.max(axis=0))
    assert np.array_equal(a, s.argmax(axis=0))                         # numpy: first maximal index
    one = rng.standard_normal((1, 4, 5)).astype(np.float32)
    m, a = oracle.best(one)
    assert np.array_equal(m, one[0]) and np.all(a == 0)


def test_local_z_literal_against_numpy_slices():
    rng = np.random.default_rng(6)
    m = rng.standard_normal((9, 13)).astype(np.float32)
    for box in (1, 3, 5, 31):                                          # 31 > the map: every box is the whole map
        z, sd = oracle.local_z(m, box, literal=True)
        h = (box - 1) // 2
        for y in range(9):
            for x in range(13):
                blk = m[max(0, y - h):y + h + 1, max(0, x - h):x + h + 1].astype(np.float64)
                ref = np.std(blk)                                      # population standard deviation
                assert sd[y, x] == pytest.approx(ref, rel=1e-12, abs=1e-15)
                assert z[y, x] == pytest.approx(float(m[y, x]) / ref if ref > 0 else 0.0, rel=1e-12)
    z, sd = oracle.local_z(m, 1, literal=True)
    assert np.all(sd == 0) and np.all(z == 0)                          # a single pixel has no spread


def test_local_z_separable_form_matches_literal():
    rng = np.random.default_rng(7)
    m = (rng.standard_normal((61, 77)) * 3 + 10).astype(np.float32)   # offset: tests the variance formula
    for box in (3, 11, 255):
        z1, s1 = oracle.local_z(m, box, literal=True)
        z2, s2 = oracle.local_z(m, box)
        assert np.max(np.abs(s1 - s2)) <= 1e-9 and np.max(np.abs(z1 - z2)) <= 1e-7


def test_local_z_closed_forms_and_invariances():
    H = W = 40
    assert np.all(oracle.local_z(np.full((H, W), 2.5, np.float32), 7)[0] == 0)      # constant map
    yy, xx = np.mgrid[0:H, 0:W]
    cb = np.where((yy + xx) % 2 == 0, 1.0, -1.0).astype(np.float32)
    n = 7
    z, sd = oracle.local_z(cb, n)
    # interior: (n^2 + 1)/2 pixels of the centre's sign, mean = +-1/n^2, variance = 1 - 1/n^4
    assert np.allclose(sd[5:-5, 5:-5], math.sqrt(1.0 - 1.0 / n ** 4), rtol=0, atol=1e-12)
    assert np.allclose(z[5:-5, 5:-5], cb[5:-5, 5:-5].astype(np.float64) / math.sqrt(1.0 - 1.0 / n ** 4), rtol=0, atol=1e-12)
    # corner (0, 0): a 4 x 4 block with 8 pixels of each sign -> variance 1
    assert sd[0, 0] == pytest.approx(1.0, abs=1e-12)
    rng = np.random.default_rng(8)
    m = rng.standard_normal((H, W)).astype(np.float32)
    z1 = oracle.local_z(m, 9)[0]
    assert np.allclose(oracle.local_z(4.0 * m, 9)[0], z1, rtol=1e-12)             # units of sigma
    assert np.allclose(oracle.local_z(-m, 9)[0], -z1, rtol=1e-12)
    assert np.allclose(oracle.local_z(m[::-1, ::-1].copy(), 9)[0], z1[::-1, ::-1], rtol=1e-12)


def test_local_sigma_of_unit_noise_is_one():
    rng = np.random.default_rng(9)
    m = rng.standard_normal((300, 300)).astype(np.float32)
    _, sd = oracle.local_z(m, 255)
    assert abs(sd[150, 150] - 1.0) < 4.0 / math.sqrt(2 * 255 * 255)
    assert abs(sd[0, 0] - 1.0) < 4.0 / math.sqrt(2 * 128 * 128)
