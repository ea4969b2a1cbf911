"""GPU parity of tno_mf_search_masked (per-pixel validity weights in D) against the oracle."""
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


def _run(f, v, sigma, traj, t0, topk, thr, generic=False, times=None, jitter=None, limit=0):
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    with MatchedFilter(0, topk, thr, generic, workspace_limit_mb=limit) as mf:
        maps, cand = mf.search(torch.from_numpy(f).cuda(), sigma, traj, 1.0, t0, frame_times=times,
                               jitter_xy=jitter, valid=torch.from_numpy(v).cuda())
        torch.cuda.synchronize()
        return maps.cpu().numpy(), mf.candidates_to_numpy(cand), mf.stats()


def _stack(shape, seed):
    rng = np.random.default_rng(seed)
    T, H, W = shape
    valid = (rng.uniform(size=shape) > 0.15).astype(np.float32)
    valid[:, H // 3:H // 3 + 6, W // 4:W // 4 + 9] = 0.0            # a masked star in every frame
    valid[T // 2] = 0.0                                             # a lost frame
    r = rng.standard_normal(shape).astype(np.float32)
    r[:, H // 2, W // 2] += 4.0
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    return (r * valid).astype(np.float32), valid, sigma


TRAJ = np.array([[0.12, -0.2, 0, 0], [0.12, 0.33, 0, 0], [0.12, 0.0, 0, 0.002], [-0.4, 0.1, 0.001, 0],
                 [0.0, 0.0, 0, 0]], np.float32)


@pytest.mark.parametrize("shape,generic", [((40, 96, 128), False), ((70, 130, 68), False), ((9, 33, 47), True),
                                           ((20, 64, 64), True)])
def test_masked_search_matches_oracle(shape, generic):
    f, v, sigma = _stack(shape, sum(shape))
    t0 = shape[0] / 2.0
    om = oracle.snr_map(f, sigma, TRAJ, 1.0, t0, valid=v)
    gm, gc, stats = _run(f, v, sigma, TRAJ, t0, 6, 3.0, generic)
    assert stats[1] == (0 if (generic or shape[2] % 4) else 1)
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
    for k in range(TRAJ.shape[0]):
        check_topk(gc[k], om[k], k, 6, 3.0)
        check_topk_vs_own_map(gc[k], gm[k], k, 6, 3.0)
    # under the masked star with a static track nothing is left: D = 0 -> SNR = 0
    H, W = shape[1], shape[2]
    assert gm[4, H // 3 + 3, W // 4 + 4] == 0.0 and om[4, H // 3 + 3, W // 4 + 4] == 0.0


def test_all_valid_agrees_with_the_plain_search_and_chunks_are_identical():
    torch = _torch()
    from helpers import run_gpu
    shape = (50, 128, 128)
    f, v, sigma = _stack(shape, 5)
    ones = np.ones_like(f)
    vs = np.linspace(-0.3, 0.3, 4).astype(np.float32)
    traj = np.array([[vx, vy, 0, 0] for vx in vs for vy in vs], np.float32)
    plain, _, _ = run_gpu(torch.from_numpy(f).cuda(), sigma, traj, 1.0, 25.0, 5, 3.0)
    masked, _, _ = _run(f, ones, sigma, traj, 25.0, 5, 3.0)
    assert np.abs(plain - masked).max() <= 2e-5 * max(1.0, float(np.abs(plain).max()))     # D analytic vs accumulated
    a, ca, sa = _run(f, v, sigma, traj, 25.0, 5, 3.0)
    b, cb, sb = _run(f, v, sigma, traj, 25.0, 5, 3.0, limit=1)                             # forced chunking
    assert sb[0] > sa[0] and np.array_equal(a, b) and np.array_equal(ca, cb)
    om = oracle.snr_map(f, sigma, traj, 1.0, 25.0, valid=v)
    assert np.abs(a.astype(np.float64) - om).max() <= TOL


def test_masked_with_times_and_jitter_and_fractional_weights():
    shape = (30, 64, 96)
    f, v, sigma = _stack(shape, 6)
    rng = np.random.default_rng(7)
    w = (v * rng.uniform(0.25, 1.0, size=shape)).astype(np.float32)          # relative inverse variances
    fw = (f * (w / np.where(v > 0, v, 1.0))).astype(np.float32)
    times = np.cumsum(rng.uniform(0.5, 1.5, shape[0])).astype(np.float32)
    jitter = rng.uniform(-1.5, 1.5, (shape[0], 2)).astype(np.float32)
    t0 = float(times[15])
    om = oracle.snr_map(fw, sigma, TRAJ, 1.0, t0, times=times, jitter=jitter, valid=w)
    gm, _, _ = _run(fw, w, sigma, TRAJ, t0, 4, 3.0, times=times, jitter=jitter)
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
