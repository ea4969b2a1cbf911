"""GPU parity of tno_mf_search_ex (frame times, pointing jitter: PAPER.md L106, L116) against the oracle."""
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


def _run(f, sigma, traj, t0, times, jitter, topk, thr, force_generic=False):
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    with MatchedFilter(0, topk, thr, force_generic) as mf:
        maps, cand = mf.search(torch.from_numpy(f).cuda(), sigma, traj, 1.0, t0, frame_times=times,
                               jitter_xy=jitter)
        torch.cuda.synchronize()
        return maps.cpu().numpy(), mf.candidates_to_numpy(cand), mf.stats()


@pytest.mark.parametrize("shape,generic", [((40, 96, 128), False), ((70, 130, 68), False), ((9, 33, 47), True),
                                           ((150, 64, 64), False)])
def test_times_and_jitter_match_oracle(shape, generic):
    T, H, W = shape
    rng = np.random.default_rng(T + H + W)
    f = rng.standard_normal(shape).astype(np.float32)
    f[:, H // 2, W // 2] += 4.0
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    # a transmission gap after the first half, irregular cadence, sub-pixel jitter with a slow drift
    times = (np.arange(T) * 1.0 + np.where(np.arange(T) >= T // 2, 11.5, 0.0) +
             rng.uniform(-0.2, 0.2, T)).astype(np.float32)
    jitter = (0.6 * rng.standard_normal((T, 2)) + np.linspace(-1.5, 1.5, T)[:, None]).astype(np.float32)
    traj = np.array([[0.12, -0.2, 0, 0], [0.12, 0.33, 0, 0], [0.12, 0.0, 0, 0.002], [-0.4, 0.1, 0.001, 0],
                     [0.0, 0.0, 0, 0]], np.float32)
    t0 = float(times[T // 2])
    om = oracle.snr_map(f, sigma, traj, 1.0, t0, times=times, jitter=jitter)
    gm, gc, stats = _run(f, sigma, traj, t0, times, jitter, 6, 3.0, generic)
    assert stats[1] == (0 if (generic or W % 4) else 1)
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
    for k in range(traj.shape[0]):
        check_topk(gc[k], om[k], k, 6, 3.0)
        check_topk_vs_own_map(gc[k], gm[k], k, 6, 3.0)
    # only one of the two given; and the plain call equals frame-index times with zero jitter
    om_t = oracle.snr_map(f, sigma, traj, 1.0, t0, times=times)
    gm_t, _, _ = _run(f, sigma, traj, t0, times, None, 6, 3.0, generic)
    assert np.abs(gm_t.astype(np.float64) - om_t).max() <= TOL
    base, _, _ = _run(f, sigma, traj, t0, None, None, 6, 3.0, generic)
    same, _, _ = _run(f, sigma, traj, t0, np.arange(T, dtype=np.float32), np.zeros((T, 2), np.float32), 6, 3.0,
                      generic)
    assert np.array_equal(base, same)


def test_injected_source_is_recovered_at_a_sqrt_d_and_bad_values_are_rejected():
    torch = _torch()
    import paper_2209_09848_b200 as P
    T, H, W = 60, 64, 64
    rng = np.random.default_rng(3)
    sigma = np.ones(T, np.float32)
    times = np.cumsum(rng.uniform(0.5, 1.5, T)).astype(np.float32)
    jitter = rng.uniform(-2, 2, (T, 2)).astype(np.float32)
    tr = np.array([[0.21, -0.13, 0, 0]], np.float32)
    t0 = float(times[30])
    f = np.zeros((T, H, W), np.float32)
    oracle.inject(f, tr, [30], [33], [1.5], 1.0, t0, times=times, jitter=jitter)
    gm, _, _ = _run(f, sigma, tr, t0, times, jitter, 3, 3.0)
    _, N, D = oracle.point(f, sigma, tr[0], 1.0, t0, 30, 33, times=times, jitter=jitter)
    assert gm[0, 33, 30] == pytest.approx(1.5 * np.sqrt(D), rel=1e-5)
    assert np.unravel_index(np.argmax(gm[0]), gm[0].shape) == (33, 30)
    ctx = P.tno_mf_create(0, None, 3, 5.0)
    d = torch.from_numpy(f).cuda()
    out = torch.empty((1, H, W), device="cuda")
    bad = times.copy(); bad[5] = np.nan
    with pytest.raises(P.TnoMfError):
        P.tno_mf_search_ex(ctx, d, sigma, bad, None, tr, 1.0, t0, out)
    badj = jitter.copy(); badj[7, 1] = np.inf
    with pytest.raises(P.TnoMfError):
        P.tno_mf_search_ex(ctx, d, sigma, None, badj, tr, 1.0, t0, out)
    P.tno_mf_destroy(ctx)


def test_injection_on_the_jittered_track_is_recovered_by_search_ex():
    """tno_mf_inject_ex renders the source on the track that tno_mf_search_ex scores (irregular cadence + jitter):
    it equals the oracle's renderer, and the search finds the source at its start pixel with SNR = A sqrt(D)."""
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    T, H, W = 50, 64, 96
    rng = np.random.default_rng(4)
    times = (np.arange(T) + np.where(np.arange(T) >= 20, 7.25, 0.0) + rng.uniform(-0.3, 0.3, T)).astype(np.float32)
    jitter = (0.7 * rng.standard_normal((T, 2))).astype(np.float32)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    tr = np.array([[0.21, -0.13, 0.001, 0.0005], [-0.3, 0.3, 0, 0]], np.float32)
    t0 = float(times[T // 2])
    ref = np.zeros((T, H, W), np.float32)
    oracle.inject(ref, tr, [40, 70], [30, 12], [6.0, 9.0], 1.0, t0, times=times, jitter=jitter)
    with MatchedFilter(0, 3, 5.0) as mf:
        d = torch.zeros((T, H, W), dtype=torch.float32, device="cuda")
        mf.inject(d, tr, [40, 70], [30, 12], [6.0, 9.0], 1.0, t0, frame_times=times, jitter_xy=jitter)
        torch.cuda.synchronize()
        assert np.array_equal(d.cpu().numpy(), ref)
        plain = torch.zeros_like(d)
        mf.inject(plain, tr, [40, 70], [30, 12], [6.0, 9.0], 1.0, t0)           # without times / jitter: another track
        assert not torch.equal(plain, d)
        maps, cand = mf.search(d, sigma, tr, 1.0, t0, frame_times=times, jitter_xy=jitter)
        torch.cuda.synchronize()
        c = mf.candidates_to_numpy(cand)
        for k, (x, y, A) in enumerate(((40, 30, 6.0), (70, 12, 9.0))):
            s, N, D = oracle.point(ref, sigma, tr[k], 1.0, t0, x, y, times=times, jitter=jitter)
            assert abs(N / D - A) < 1e-4 * A and abs(s - A * np.sqrt(D)) < 1e-4 * s
            assert (int(c[k]["x"][0]), int(c[k]["y"][0])) == (x, y) and abs(float(c[k]["snr"][0]) - s) <= TOL
        with pytest.raises(P.TnoMfError):                   # a displacement beyond 32-bit pixel arithmetic
            mf.inject(d, np.array([[3e8, 0, 0, 0]], np.float32), [1], [1], [1.0], 1.0, 0.0)
        bad = times.copy(); bad[3] = np.nan
        with pytest.raises(P.TnoMfError):
            mf.inject(d, tr, [40, 70], [30, 12], [6.0, 9.0], 1.0, t0, frame_times=bad)
