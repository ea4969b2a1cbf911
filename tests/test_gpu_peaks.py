"""GPU parity of tno_mf_peaks (non-maximum suppression of a score map) against the oracle:
exact (comparisons only), including ties, frame borders, thresholds and the candidate list; and the point of it:
one injected object gives one candidate."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _check(score, radius, topk=6, thr=1.0, argk=None):
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    score = np.ascontiguousarray(score, dtype=np.float32)
    with MatchedFilter(0, topk, thr) as mf:
        d = torch.from_numpy(score).cuda()
        a = torch.from_numpy(argk).cuda() if argk is not None else None
        pk, top = mf.peaks(d, radius, a)
        torch.cuda.synchronize()
        pk = pk.cpu().numpy()
        c = mf.candidates_to_numpy(top[None])[0]
    keep = oracle.peaks(score, radius, thr)
    assert np.array_equal(np.isfinite(pk) | (pk == np.inf), keep)
    assert np.array_equal(pk[keep], score[keep]) and np.all(pk[~keep] == -np.inf)
    ref = oracle.topk(np.where(keep, score.astype(np.float64), -np.inf), topk, max(thr, -3e38), 0)
    assert np.array_equal(c["x"], ref["x"]) and np.array_equal(c["y"], ref["y"])
    assert np.array_equal(c["snr"].astype(np.float64), ref["snr"])
    n = int(np.count_nonzero(c["x"] >= 0))
    if argk is not None:
        assert np.array_equal(c["k"][:n], argk[c["y"][:n], c["x"][:n]]) and np.all(c["k"][n:] == -1)
    return c, n


@pytest.mark.parametrize("shape,radius", [((64, 64), 2), ((70, 132), 5), ((33, 47), 1), ((300, 260), 12), ((1, 1), 3),
                                          ((513, 17), 0), ((5, 200), 40)])
def test_peaks_match_oracle(shape, radius):
    rng = np.random.default_rng(sum(shape) + radius)
    _check(rng.standard_normal(shape), radius, argk=rng.integers(0, 9, shape).astype(np.int32))


def test_ties_thresholds_and_errors():
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    rng = np.random.default_rng(4)
    _check(rng.integers(0, 4, (40, 48)), 2)                                  # plateaus: first in row-major order
    _check(np.full((32, 32), 1.5), 3)                                        # constant map: pixel (0, 0) and every
    c, n = _check(rng.standard_normal((50, 50)), 4, topk=1000, thr=-np.inf)  # no threshold, list longer than peaks
    assert 0 < n < 1000
    _, n = _check(rng.standard_normal((20, 20)), 2, thr=50.0)                # nothing above the threshold
    assert n == 0
    with MatchedFilter(0, 4, 0.0) as mf:
        d = torch.zeros((8, 8), device="cuda")
        for bad in (-1, 5000):
            with pytest.raises(P.TnoMfError):
                P.tno_mf_peaks(mf.ctx, d, None, bad, torch.empty_like(d), None)
        with pytest.raises(P.TnoMfError):
            P.tno_mf_peaks(mf.ctx, d, None, 2, d, None)                      # aliasing
        with pytest.raises(P.TnoMfError):
            P.tno_mf_peaks(mf.ctx, d, None, 2, None, None)                   # no output


def test_one_object_one_candidate():
    """An injected mover lights up a neighbourhood of start pixels and several neighbouring trajectories: without
    suppression the top of the list is that one object many times over; with it, once."""
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    rng = np.random.default_rng(7)
    T, H, W = 120, 96, 128
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    trajs = np.array([[vx, vy, 0, 0] for vx in (0.10, 0.15, 0.20) for vy in (-0.05, 0.0, 0.05)], np.float32)
    oracle.inject(f, trajs[4:5], [60], [40], [1.2], 1.0, T / 2.0)
    with MatchedFilter(0, 10, 5.0) as mf:
        maps, _ = mf.search(torch.from_numpy(f).cuda(), np.ones(T, np.float32), trajs, 1.0, T / 2.0)
        mx, ak, z, top = mf.best(maps, 63)
        pk, ptop = mf.peaks(z, 5, ak)
        torch.cuda.synchronize()
        raw = mf.candidates_to_numpy(top[None])[0]
        nms = mf.candidates_to_numpy(ptop[None])[0]
    assert np.count_nonzero(raw["x"] >= 0) >= 5                 # the same object, many pixels
    assert np.count_nonzero(nms["x"] >= 0) == 1
    assert abs(int(nms["x"][0]) - 60) <= 1 and abs(int(nms["y"][0]) - 40) <= 1 and int(nms["k"][0]) == 4
