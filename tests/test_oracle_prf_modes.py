"""Pins for the oracle's pixel-integrated Gaussian (filter 2) and tabulated PRF (filter 3) -- SURVEY 8(f) rank 3,
PAPER.md:L41 (the PRF as the fraction of the flux per pixel: ~50 % in the peak pixel, ~90 % in 2 x 2).
Each check uses something the oracle does not compute itself: numerical quadrature of the Gaussian density,
closed-form limits, an explicit numpy evaluation of the definition with a hand-made table."""
import numpy as np
import scipy.integrate

import oracle


def _one_frame_taps(filter, prf_sigma, phase_x, phase_y, prf_table=None, size=9):
    """The 2-D filter of one frame at sub-pixel offset (phase_x, phase_y), read off the oracle: N of a stack
    that is 1 at a single pixel, for the trajectory that is displaced by the phase (T = 1, q = 1)."""
    c = size // 2
    out = np.zeros((size, size))
    traj = np.array([phase_x, phase_y, 0, 0], np.float32)
    for py in range(size):
        for px in range(size):
            f = np.zeros((1, size, size), np.float32)
            f[0, py, px] = 1.0
            # frame time 1 with t0 = 0: displacement = (phase_x, phase_y)
            _, N, _ = oracle.point(f, [1.0], traj, prf_sigma, 0.0, c, c, times=np.array([1.0], np.float32),
                                   filter=filter, prf_table=prf_table)
            out[py, px] = N
    return out


def test_pixel_integrated_taps_equal_quadrature_of_the_gaussian_density():
    s = float(np.float32(0.8))           # prf_sigma crosses the boundary as float32
    for phx, phy in ((0.0, 0.0), (0.3, -0.45), (-0.5, 0.25)):
        phx32, phy32 = float(np.float32(phx)), float(np.float32(phy))
        g = _one_frame_taps(2, s, phx, phy)
        c = 4
        for j in range(-2, 3):
            for i in range(-2, 3):
                dens = lambda y, x: np.exp(-((x - phx32) ** 2 + (y - phy32) ** 2) / (2 * s * s)) / (2 * np.pi * s * s)
                ref, _ = scipy.integrate.dblquad(dens, i - 0.5, i + 0.5, j - 0.5, j + 0.5, epsabs=1e-12)
                assert abs(g[c + j, c + i] - ref) < 1e-9, (i, j, g[c + j, c + i], ref)
        # nothing outside the 5 x 5 window
        mask = np.ones_like(g, bool)
        mask[c - 2:c + 3, c - 2:c + 3] = False
        assert np.all(g[mask] == 0)


def test_pixel_integrated_flux_fractions():
    """Closed forms: the taps of one axis sum to Phi((2.5-ph)/s) - Phi((-2.5-ph)/s) (~1: the window holds the
    flux); a narrow PRF puts everything into the rounded pixel (the shift-stack filter); a centred source of
    sigma s has erf(1/(2 sqrt 2 s))^2 of its flux in the peak pixel."""
    from math import erf, sqrt
    s = float(np.float32(0.7))           # prf_sigma crosses the boundary as float32
    g = _one_frame_taps(2, s, 0.2, -0.1)
    ph = float(np.float32(0.2)), float(np.float32(-0.1))
    Phi = lambda z: 0.5 * (1 + erf(z / sqrt(2)))
    fx = Phi((2.5 - ph[0]) / s) - Phi((-2.5 - ph[0]) / s)
    fy = Phi((2.5 - ph[1]) / s) - Phi((-2.5 - ph[1]) / s)
    assert abs(g.sum() - fx * fy) < 1e-12 and g.sum() > 0.999
    narrow = _one_frame_taps(2, 0.02, 0.3, 0.3)
    stack = _one_frame_taps(1, 0.02, 0.3, 0.3)
    assert np.allclose(narrow, stack, atol=1e-12) and stack.sum() == 1.0
    centred = _one_frame_taps(2, s, 0.0, 0.0)
    assert abs(centred[4, 4] - erf(1 / (2 * sqrt(2) * s)) ** 2) < 1e-12
    # the paper's PRF (L41): ~50 % of the flux in the peak pixel <=> erf(1 / (2 sqrt2 s)) = sqrt(1/2), s = 0.4754 px
    assert abs(_one_frame_taps(2, 0.4754, 0.0, 0.0)[4, 4] - 0.5) < 1e-3


def test_tabulated_prf_reads_the_row_of_the_phase():
    rng = np.random.default_rng(3)
    n_phase = 8
    tab = rng.uniform(0.0, 1.0, (n_phase, 5))
    for phx, phy in ((-0.5, 0.49), (0.0, 0.124), (0.126, -0.3)):
        g = _one_frame_taps(3, 1.0, phx, phy, prf_table=tab)
        rx = min(n_phase - 1, int(np.floor((float(np.float32(phx)) + 0.5) * n_phase)))
        ry = min(n_phase - 1, int(np.floor((float(np.float32(phy)) + 0.5) * n_phase)))
        assert np.allclose(g[2:7, 2:7], np.outer(tab[ry], tab[rx]), rtol=0, atol=1e-15)


def test_map_and_point_agree_and_injected_source_is_recovered_in_every_mode():
    """snr_map (separable evaluation) equals point (literal 25 taps); a noiseless source injected with the mode's
    own PRF gives N / D = its amplitude at its start pixel (the matched filter is the ML flux estimate, L108)."""
    rng = np.random.default_rng(11)
    T, H, W = 12, 20, 24
    sigma_t = rng.uniform(0.8, 1.3, T).astype(np.float32)
    trajs = np.array([[0.31, -0.22, 0.004, 0.002], [-0.4, 0.15, 0.0, -0.003]], np.float32)
    phases = 16
    u = np.arange(-2, 3)[None, :] - ((np.arange(phases) + 0.5) / phases - 0.5)[:, None]
    tab = np.exp(-np.abs(u) / 0.6)
    tab /= tab.sum(axis=1, keepdims=True)
    for mode, table in ((2, None), (3, tab)):
        frames = rng.standard_normal((T, H, W)).astype(np.float32)
        m = oracle.snr_map(frames, sigma_t, trajs, 0.9, 5.0, filter=mode, prf_table=table)
        for k, x, y in ((0, 3, 4), (1, 12, 9), (0, 23, 19), (1, 0, 0)):
            s, _, _ = oracle.point(frames, sigma_t, trajs[k], 0.9, 5.0, x, y, filter=mode, prf_table=table)
            assert abs(m[k, y, x] - s) < 1e-11
        clean = np.zeros((T, H, W), np.float32)
        oracle.inject(clean, trajs[:1], [11], [10], [37.5], 0.9, 5.0, filter=mode, prf_table=table)
        _, N, D = oracle.point(clean, sigma_t, trajs[0], 0.9, 5.0, 11, 10, filter=mode, prf_table=table)
        assert abs(N / D - 37.5) < 1e-4


# ---- filter 4: tabulated NON-separable PRF ------------------------------------------
def _table2d(rng, ny, nx):
    """A random non-negative [ny, nx, 5, 5] table that is NOT an outer product (rank > 1 blocks)."""
    tab = rng.uniform(0.0, 1.0, (ny, nx, 5, 5))
    tab[..., 2, 2] += 2.0
    assert np.linalg.matrix_rank(tab[0, 0]) > 1
    return tab


def test_nonseparable_table_reads_the_block_of_both_phases():
    """An explicit 25-tap lookup: the frame's filter is the 5 x 5 block at (row of the y-phase, column of the
    x-phase), entry [j + 2][i + 2] at pixel offset (i, j) -- transposing the block, swapping the phase axes or
    mirroring a tap index fails (the table is random, with ny != nx)."""
    rng = np.random.default_rng(7)
    ny, nx = 6, 4
    tab = _table2d(rng, ny, nx)
    for phx, phy in ((-0.5, 0.49), (0.0, 0.124), (0.126, -0.3), (0.3, 0.3)):
        g = _one_frame_taps(4, 1.0, phx, phy, prf_table=tab)
        rx = min(nx - 1, int(np.floor((float(np.float32(phx)) + 0.5) * nx)))
        ry = min(ny - 1, int(np.floor((float(np.float32(phy)) + 0.5) * ny)))
        assert np.array_equal(g[2:7, 2:7], tab[ry, rx])           # g[row = y offset + 2, column = x offset + 2]
        mask = np.ones_like(g, bool)
        mask[2:7, 2:7] = False
        assert np.all(g[mask] == 0)


def test_nonseparable_table_of_outer_products_is_the_separable_mode():
    """Reduction to mode 3: with table2d[ry, rx] = outer(tab[ry], tab[rx]) maps, N and D are those of the separable
    tabulated filter (same products, so equal to rounding of one multiplication)."""
    rng = np.random.default_rng(5)
    n_phase = 8
    tab = rng.uniform(0.1, 1.0, (n_phase, 5))
    tab2 = np.einsum("yj,xi->yxji", tab, tab)
    T, H, W = 9, 14, 17
    frames = rng.standard_normal((T, H, W)).astype(np.float32)
    sigma_t = rng.uniform(0.8, 1.3, T).astype(np.float32)
    trajs = np.array([[0.31, -0.22, 0.004, 0.002], [-0.4, 0.15, 0.0, -0.003], [0.5, 0.25, 0, 0]], np.float32)
    m3, N3, D3 = oracle.snr_map(frames, sigma_t, trajs, 1.0, 4.0, filter=3, prf_table=tab, return_ND=True)
    m4, N4, D4 = oracle.snr_map(frames, sigma_t, trajs, 1.0, 4.0, filter=4, prf_table=tab2, return_ND=True)
    assert np.allclose(N4, N3, rtol=1e-13, atol=1e-13) and np.allclose(D4, D3, rtol=1e-13, atol=0)
    assert np.allclose(m4, m3, rtol=1e-12, atol=1e-12)


def test_nonseparable_map_point_brute_force_and_injection():
    """snr_map (hoisted) equals point (literal) in mode 4; both equal a Python evaluation of the definition written
    out here (exact-rational displacement, explicit table lookup, off-frame taps dropped from N and D); a noiseless
    source injected with the same table gives N / D = its amplitude."""
    from fractions import Fraction
    import math
    rng = np.random.default_rng(13)
    ny, nx = 5, 7
    tab = _table2d(rng, ny, nx)
    T, H, W = 6, 9, 11
    frames = rng.standard_normal((T, H, W)).astype(np.float32)
    sigma_t = rng.uniform(0.8, 1.3, T).astype(np.float32)
    trajs = np.array([[0.31, -0.22, 0.01, 0.02], [-0.9, 0.55, 0.0, -0.03]], np.float32)
    t0 = 2.0
    m = oracle.snr_map(frames, sigma_t, trajs, 1.0, t0, filter=4, prf_table=tab)

    def brute(k, x, y):
        N = D = 0.0
        for t in range(T):
            dt = Fraction(t) - Fraction(t0)
            d = [Fraction(float(trajs[k, a])) * dt + Fraction(float(trajs[k, a + 2])) * dt * dt for a in (0, 1)]
            s = [math.floor(v + Fraction(1, 2)) for v in d]
            ph = [float(v - sv) for v, sv in zip(d, s)]
            rx = min(nx - 1, max(0, math.floor((ph[0] + 0.5) * nx)))
            ry = min(ny - 1, max(0, math.floor((ph[1] + 0.5) * ny)))
            q = 1.0 / float(sigma_t[t]) ** 2
            for j in range(-2, 3):
                for i in range(-2, 3):
                    px, py = x + s[0] + i, y + s[1] + j
                    if 0 <= px < W and 0 <= py < H:
                        g = tab[ry, rx, j + 2, i + 2]
                        N += g * float(frames[t, py, px]) * q
                        D += g * g * q
        return N / math.sqrt(D) if D > 0 else 0.0

    for k, x, y in ((0, 3, 4), (1, 7, 2), (0, 10, 8), (1, 0, 0), (0, 0, 8)):
        s, _, _ = oracle.point(frames, sigma_t, trajs[k], 1.0, t0, x, y, filter=4, prf_table=tab)
        assert abs(m[k, y, x] - s) < 1e-11
        assert abs(s - brute(k, x, y)) < 1e-11
    clean = np.zeros((T, H, W), np.float32)
    oracle.inject(clean, trajs[:1], [5], [4], [21.5], 1.0, t0, filter=4, prf_table=tab)
    _, N, D = oracle.point(clean, sigma_t, trajs[0], 1.0, t0, 5, 4, filter=4, prf_table=tab)
    assert abs(N / D - 21.5) < 1e-5
