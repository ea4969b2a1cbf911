"""GPU parity of the pixel-integrated Gaussian (cfg.filter = 2) and the tabulated separable PRF (cfg.filter = 3,
tno_mf_set_prf_table) against the oracle: maps, candidate lists, injection, flux, error paths."""
import numpy as np
import pytest

import oracle
from helpers import TOL, check_topk, check_topk_vs_own_map

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _table(n_phase, width=0.6):
    """An exponential-profile PRF, normalised per phase: nothing like a Gaussian on purpose."""
    u = np.arange(-2, 3)[None, :] - ((np.arange(n_phase) + 0.5) / n_phase - 0.5)[:, None]
    tab = np.exp(-np.abs(u) / width)
    return (tab / tab.sum(axis=1, keepdims=True)).astype(np.float32)


TRAJ = np.array([[0.12, -0.2, 0, 0], [0.12, 0.33, 0, 0], [0.12, 0.0, 0, 0.002], [-0.4, 0.1, 0.001, 0],
                 [0.0, 0.0, 0, 0]], np.float32)


@pytest.mark.parametrize("mode", [2, 3])
@pytest.mark.parametrize("shape,generic", [((40, 96, 128), False), ((9, 33, 47), True), ((70, 130, 68), False)])
def test_maps_and_lists_match_oracle(mode, shape, generic):
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    T, H, W = shape
    rng = np.random.default_rng(sum(shape) + mode)
    f = rng.standard_normal(shape).astype(np.float32)
    f[:, H // 2, W // 2] += 3.0
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    tab = _table(11) if mode == 3 else None
    jit = (0.3 * rng.standard_normal((T, 2))).astype(np.float32)
    om = oracle.snr_map(f, sigma, TRAJ, 0.7, T / 2.0, jitter=jit, filter=mode, prf_table=tab)
    with MatchedFilter(0, 5, 3.0, generic, filter=mode, prf_table=tab) as mf:
        maps, cand = mf.search(torch.from_numpy(f).cuda(), sigma, TRAJ, 0.7, T / 2.0, jitter_xy=jit)
        torch.cuda.synchronize()
        assert mf.stats()[1] == (0 if (generic or W % 4) else 1)
        gm, gc = maps.cpu().numpy(), mf.candidates_to_numpy(cand)
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
    for k in range(TRAJ.shape[0]):
        check_topk(gc[k], om[k], k, 5, 3.0)
        check_topk_vs_own_map(gc[k], gm[k], k, 5, 3.0)


@pytest.mark.parametrize("mode", [2, 3])
def test_injection_and_flux_use_the_modes_prf(mode):
    """tno_mf_inject renders with the taps of the mode (oracle.inject, within one float32 ulp: erf / table values
    are rounded in double on both sides); the flux estimate of the source is its amplitude."""
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    T, H, W = 60, 64, 64
    tab = _table(16) if mode == 3 else None
    tr = np.array([[0.137, -0.081, 0.0005, 0]], np.float32)
    ref = np.zeros((T, H, W), np.float32)
    oracle.inject(ref, tr, [32], [30], [25.0], 0.6, 30.0, filter=mode, prf_table=tab)
    with MatchedFilter(0, filter=mode, prf_table=tab) as mf:
        d = torch.zeros((T, H, W), dtype=torch.float32, device="cuda")
        mf.inject(d, tr, [32], [30], [25.0], 0.6, 30.0)
        torch.cuda.synchronize()
        got = d.cpu().numpy()
        assert np.abs(got - ref).max() <= 2e-6 * 25.0 and got.sum() > 0.99 * 25.0 * T
        maps, _ = mf.search(d, np.ones(T, np.float32), tr, 0.6, 30.0)
        flux = mf.flux(maps)
        torch.cuda.synchronize()
        assert abs(float(flux[0, 30, 32]) - 25.0) < 1e-3 * 25.0


def test_pixel_integrated_differs_from_point_sampled_and_errors():
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    rng = np.random.default_rng(1)
    T, H, W = 30, 32, 64
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    sigma = np.ones(T, np.float32)
    d = torch.from_numpy(f).cuda()
    with MatchedFilter(0) as a, MatchedFilter(0, filter=2) as b:
        ma, _ = a.search(d, sigma, TRAJ[:2], 0.5, 15.0)
        mb, _ = b.search(d, sigma, TRAJ[:2], 0.5, 15.0)
        torch.cuda.synchronize()
        assert float((ma - mb).abs().max()) > 0.05          # a narrow PRF: sampling and integrating differ
    with pytest.raises(P.TnoMfError):
        P.tno_mf_create(0, filter=5)
    with MatchedFilter(0, filter=3) as c:
        with pytest.raises(P.TnoMfError):                   # no table yet
            c.search(d, sigma, TRAJ[:2], 0.5, 15.0)
        with pytest.raises(P.TnoMfError):
            P.tno_mf_set_prf_table(c.ctx, np.array([[0.1, 0.2, np.nan, 0.2, 0.1]], np.float32))
        with pytest.raises(P.TnoMfError):
            P.tno_mf_set_prf_table(c.ctx, np.array([[0.1, 0.2, -0.4, 0.2, 0.1]], np.float32))
        P.tno_mf_set_prf_table(c.ctx, _table(4))
        m1, _ = c.search(d, sigma, TRAJ[:2], 0.5, 15.0)
        om = oracle.snr_map(f, sigma, TRAJ[:2], 0.5, 15.0, filter=3, prf_table=_table(4))
        torch.cuda.synchronize()
        assert np.abs(m1.cpu().numpy() - om).max() <= TOL
        P.tno_mf_set_prf_table(c.ctx, None)                 # removed again
        with pytest.raises(P.TnoMfError):
            c.search(d, sigma, TRAJ[:2], 0.5, 15.0)


# ---- filter 4: tabulated non-separable PRF (tno_mf_set_prf_table2d) ------------------
def _table2d(ny, nx, seed=0):
    """A PRF that is NOT an outer product: an elliptical, rotated exponential profile sampled per 2-D phase, plus
    a little seeded structure; normalised to unit flux per phase."""
    rng = np.random.default_rng(seed)
    phy = ((np.arange(ny) + 0.5) / ny - 0.5)[:, None, None, None]
    phx = ((np.arange(nx) + 0.5) / nx - 0.5)[None, :, None, None]
    j = np.arange(-2, 3)[None, None, :, None] - phy
    i = np.arange(-2, 3)[None, None, None, :] - phx
    u, v = 0.8 * i + 0.6 * j, -0.6 * i + 0.8 * j                    # rotated axes: couples x and y
    tab = np.exp(-np.sqrt((u / 0.9) ** 2 + (v / 0.5) ** 2)) * (1.0 + 0.1 * rng.uniform(size=(ny, nx, 5, 5)))
    tab /= tab.sum(axis=(2, 3), keepdims=True)
    assert np.linalg.matrix_rank(tab[0, 0]) > 1
    return tab.astype(np.float32)


@pytest.mark.parametrize("shape,masked", [((16, 64, 64), False), ((100, 256, 256), False), ((9, 33, 47), True),
                                          ((40, 96, 128), True)])
def test_nonseparable_prf_maps_and_lists_match_oracle(shape, masked):
    """Config-1 and config-2 shapes (and two ragged ones) with pointing jitter, with and without validity weights."""
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    T, H, W = shape
    rng = np.random.default_rng(sum(shape))
    f = rng.standard_normal(shape).astype(np.float32)
    f[:, H // 2, W // 2] += 3.0
    valid = (rng.uniform(size=shape) > 0.04).astype(np.float32) if masked else None
    if masked:
        f *= valid
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    tab = _table2d(7, 5, seed=T)
    jit = (0.3 * rng.standard_normal((T, 2))).astype(np.float32)
    om = oracle.snr_map(f, sigma, TRAJ, 1.0, T / 2.0, jitter=jit, valid=valid, filter=4, prf_table=tab)
    with MatchedFilter(0, 5, 3.0, filter=4, prf_table=tab) as mf:
        d = torch.from_numpy(f).cuda()
        maps = torch.empty((TRAJ.shape[0], H, W), device="cuda")
        cand = torch.empty((TRAJ.shape[0], 5, 4), dtype=torch.int32, device="cuda")
        P.tno_mf_search_masked(mf.ctx, d, torch.from_numpy(valid).cuda() if masked else None, sigma, None, jit, TRAJ,
                               1.0, T / 2.0, maps, cand)
        torch.cuda.synchronize()
        assert mf.stats()[1] == 0                      # the 25-tap formulation, never the separable kernel
        gm, gc = maps.cpu().numpy(), mf.candidates_to_numpy(cand)
        with pytest.raises(P.TnoMfError):              # no analytic separable D to divide by
            mf.flux(maps)
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
    for k in range(TRAJ.shape[0]):
        check_topk(gc[k], om[k], k, 5, 3.0)
        check_topk_vs_own_map(gc[k], gm[k], k, 5, 3.0)


def test_nonseparable_prf_injection_recovery_and_errors():
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    T, H, W = 60, 64, 64
    tab = _table2d(8, 8, seed=3)
    tr = np.array([[0.137, -0.081, 0.0005, 0]], np.float32)
    ref = np.zeros((T, H, W), np.float32)
    oracle.inject(ref, tr, [32], [30], [25.0], 1.0, 30.0, filter=4, prf_table=tab)
    with MatchedFilter(0, filter=4, prf_table=tab) as mf:
        d = torch.zeros((T, H, W), dtype=torch.float32, device="cuda")
        mf.inject(d, tr, [32], [30], [25.0], 1.0, 30.0)
        torch.cuda.synchronize()
        got = d.cpu().numpy()
        assert np.abs(got - ref).max() <= 2e-6 * 25.0 and got.sum() > 0.99 * 25.0 * T
        # the injected source is where the oracle puts it, with the oracle's score: SNR = A sqrt(D)
        maps, _ = mf.search(d, np.ones(T, np.float32), tr, 1.0, 30.0)
        torch.cuda.synchronize()
        s, N, D = oracle.point(ref, np.ones(T, np.float32), tr[0], 1.0, 30.0, 32, 30, filter=4, prf_table=tab)
        assert abs(N / D - 25.0) < 1e-4 and abs(float(maps[0, 30, 32]) - s) <= TOL
        assert int(maps[0].argmax()) == 30 * W + 32
        # an outer-product table gives the separable mode's maps
        t1 = _table(6)
        t2 = np.einsum("yj,xi->yxji", t1, t1).astype(np.float32)
        P.tno_mf_set_prf_table2d(mf.ctx, t2)
        f = np.random.default_rng(2).standard_normal((T, H, W)).astype(np.float32)
        m4, _ = mf.search(torch.from_numpy(f).cuda(), np.ones(T, np.float32), TRAJ, 1.0, 30.0)
        with MatchedFilter(0, filter=3, prf_table=t1) as sep:
            m3, _ = sep.search(torch.from_numpy(f).cuda(), np.ones(T, np.float32), TRAJ, 1.0, 30.0)
            torch.cuda.synchronize()
            assert float((m4 - m3).abs().max()) <= 2e-4
        with pytest.raises(P.TnoMfError):
            P.tno_mf_set_prf_table2d(mf.ctx, -t2)
        with pytest.raises(P.TnoMfError):
            bad = t2.copy(); bad[0, 0, 0, 0] = np.inf
            P.tno_mf_set_prf_table2d(mf.ctx, bad)
        P.tno_mf_set_prf_table2d(mf.ctx, None)
        with pytest.raises(P.TnoMfError):              # filter 4 without a table
            mf.search(d, np.ones(T, np.float32), tr, 1.0, 30.0)
