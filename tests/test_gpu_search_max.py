"""tno_mf_search_max: the max over the filter bank fused into the search.  The fused maps must be
bit for bit what tno_mf_best computes from the per-trajectory maps of the same search (comparisons only), on the
separable and the generic kernel, with chunked workspaces, masks, and with no other output at all; and within the
search tolerance of the oracle's maps."""
import numpy as np
import pytest

import oracle
from helpers import TOL

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _bank(n, seed):
    rng = np.random.default_rng(seed)
    vx = rng.choice([-0.3, -0.1, 0.12, 0.25], n)
    vy = rng.uniform(-0.3, 0.3, n)
    return np.stack([vx, vy, np.zeros(n), rng.choice([0.0, 0.002], n)], axis=1).astype(np.float32)


@pytest.mark.parametrize("shape,n,generic,limit_mb", [((40, 96, 128), 7, False, 0), ((9, 33, 47), 5, True, 0),
                                                      ((30, 130, 68), 23, False, 1), ((25, 64, 64), 12, True, 0)])
def test_fused_max_equals_best_of_the_maps(shape, n, generic, limit_mb):
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    T, H, W = shape
    rng = np.random.default_rng(sum(shape))
    f = rng.standard_normal(shape).astype(np.float32)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = _bank(n, n)
    d = torch.from_numpy(f).cuda()
    with MatchedFilter(0, 4, 2.5, generic, workspace_limit_mb=limit_mb) as mf:
        mx, ak, maps, top = mf.search_max(d, sigma, traj, 1.0, T / 2.0, want_maps=True)
        bm, ba, _, _ = mf.best(maps, 9)
        maps2, top2 = mf.search(d, sigma, traj, 1.0, T / 2.0)
        torch.cuda.synchronize()
        assert torch.equal(maps, maps2) and torch.equal(top, top2)          # the other outputs are unchanged
        assert torch.equal(mx, bm) and torch.equal(ak, ba)
        om, oa = oracle.best(maps.cpu().numpy())
        assert np.array_equal(mx.cpu().numpy(), om) and np.array_equal(ak.cpu().numpy(), oa)
    # no maps, no lists: the max map alone
    with MatchedFilter(0, 0, force_generic=generic, workspace_limit_mb=limit_mb) as mf:
        mx2, ak2, none_maps, none_top = mf.search_max(d, sigma, traj, 1.0, T / 2.0)
        torch.cuda.synchronize()
        assert none_maps is None and none_top is None
        assert torch.equal(mx2, mx) and torch.equal(ak2, ak)
    # against the oracle's float64 maps
    ref = oracle.snr_map(f, sigma, traj, 1.0, T / 2.0).max(axis=0)
    assert np.abs(mx.cpu().numpy().astype(np.float64) - ref).max() <= TOL


def test_ties_masks_and_errors():
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    T, H, W = 20, 64, 64
    traj = _bank(9, 3)
    sigma = np.ones(T, np.float32)
    zeros = torch.zeros((T, H, W), device="cuda")
    rng = np.random.default_rng(5)
    f = torch.from_numpy(rng.standard_normal((T, H, W)).astype(np.float32)).cuda()
    valid = torch.from_numpy((rng.uniform(size=(T, H, W)) > 0.1).astype(np.float32)).cuda()
    with MatchedFilter(0, 3, 1.0) as mf:
        mx, ak, _, _ = mf.search_max(zeros, sigma, traj, 1.0, 10.0)
        torch.cuda.synchronize()
        assert float(mx.abs().max()) == 0.0 and int(ak.max()) == 0           # all scores equal: the smallest k
        mx, ak, maps, _ = mf.search_max(f * valid, sigma, traj, 1.0, 10.0, want_maps=True, valid=valid)
        bm, ba, _, _ = mf.best(maps, 9)
        torch.cuda.synchronize()
        assert torch.equal(mx, bm) and torch.equal(ak, ba)
        with pytest.raises(P.TnoMfError):
            P.tno_mf_search_max(mf.ctx, f, None, sigma, None, None, traj, float("nan"), 10.0, mx, ak)
