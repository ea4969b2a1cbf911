"""GPU parity of the shift-stack filter mode (cfg.filter = 1) against the oracle, and the
paper's comparison: the matched filter recovers an injected source at about twice the shift-stack SNR."""
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


def _run(f, sigma, traj, t0, shift_stack, generic=False, topk=5, thr=3.0):
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    with MatchedFilter(0, topk, thr, generic, shift_stack=shift_stack) as mf:
        maps, cand = mf.search(torch.from_numpy(f).cuda(), sigma, traj, 1.0, t0)
        torch.cuda.synchronize()
        return maps.cpu().numpy(), mf.candidates_to_numpy(cand), mf.stats()


@pytest.mark.parametrize("shape,generic", [((40, 96, 128), False), ((9, 33, 47), True), ((70, 130, 68), False)])
def test_shift_stack_matches_oracle(shape, generic):
    T, H, W = shape
    rng = np.random.default_rng(sum(shape))
    f = rng.standard_normal(shape).astype(np.float32)
    f[:, H // 2, W // 2] += 3.0
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.array([[0.12, -0.2, 0, 0], [0.12, 0.33, 0, 0], [0.12, 0.0, 0, 0.002], [-0.4, 0.1, 0.001, 0],
                     [0.0, 0.0, 0, 0]], np.float32)
    om = oracle.snr_map(f, sigma, traj, 1.0, T / 2.0, shift_stack=True)
    gm, gc, stats = _run(f, sigma, traj, T / 2.0, True, generic)
    assert stats[1] == (0 if (generic or W % 4) else 1)
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
    for k in range(traj.shape[0]):
        check_topk(gc[k], om[k], k, 5, 3.0)
        check_topk_vs_own_map(gc[k], gm[k], k, 5, 3.0)


def test_matched_filter_against_shift_stack_on_an_injected_source():
    T, H, W = 200, 64, 64
    rng = np.random.default_rng(2)
    sigma = np.ones(T, np.float32)
    tr = np.array([[0.137, -0.081, 0, 0]], np.float32)
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    oracle.inject(f, tr, [32], [30], [1.0], 1.0, 100.0)
    mf_map, _, _ = _run(f, sigma, tr, 100.0, False)
    ss_map, _, _ = _run(f, sigma, tr, 100.0, True)
    # expected: A sqrt(D) ~ sqrt(200 pi) = 25 for the matched filter, ~ 0.92 sqrt(200) = 13 for shift-stack
    assert 20 < mf_map[0, 30, 32] < 30 and 8 < ss_map[0, 30, 32] < 18
    assert 1.5 < mf_map[0, 30, 32] / ss_map[0, 30, 32] < 2.4
    # both maps are unit-variance noise away from the source
    assert abs(np.std(mf_map[0, :20]) - 1.0) < 0.1 and abs(np.std(ss_map[0, :20]) - 1.0) < 0.1
