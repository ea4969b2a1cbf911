"""GPU parity of tno_mf_background (section 3.1: per-pixel Huber fit on the jitter basis) against
the float64 oracle, through the C ABI."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _case(seed, T, H, W):
    rng = np.random.default_rng(seed)
    jit = (0.4 * rng.standard_normal((T, 2)) + np.linspace(-0.3, 0.3, T)[:, None]).astype(np.float32)
    phi = oracle.background_basis(jit)
    beta = rng.standard_normal((6, H, W)) * np.array([50, 5, 5, 2, 2, 2])[:, None, None]
    y = np.einsum("tk,khw->thw", phi, beta) + 0.5 * rng.standard_normal((T, H, W))
    hit = rng.uniform(size=y.shape) < 0.03
    y = y + hit * rng.laplace(0, 20, size=y.shape)
    return y.astype(np.float32), jit


@pytest.mark.parametrize("shape,delta,n_iter", [((60, 33, 47), 1.0, 8), ((200, 64, 64), 1.5, 4), ((16, 5, 9), 1e9, 0),
                                                ((7, 1, 1), 0.5, 3), ((120, 40, 72), 0.8, 25),
                                                # staged kernel (H*W % 4 == 0): T not a multiple of the 8 frames
                                                # of a stage, T below one stage, ragged last CTA, one short CTA
                                                ((61, 36, 52), 1.2, 6), ((7, 16, 20), 0.7, 4), ((27, 4, 132), 2.0, 0),
                                                ((9, 2, 2), 0.5, 2)])
def test_background_matches_oracle(shape, delta, n_iter):
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    y, jit = _case(sum(shape), *shape)
    ob, orr = oracle.background(y, jit, delta, n_iter)
    with MatchedFilter(0) as mf:
        d = torch.from_numpy(y).cuda()
        coef, res = mf.background(d, jit, delta, n_iter)
        torch.cuda.synchronize()
        assert mf.stats()[0] == 1
        scale = float(np.abs(y).max())
        assert np.abs(res.cpu().numpy() - orr).max() <= 2e-5 * scale
        assert np.abs(coef.cpu().numpy() - ob).max() <= 2e-4 * scale        # R^-1 amplifies float32 rounding
        # in place: the residuals overwrite the stack, same values
        coef2, res2 = mf.background(d, jit, delta, n_iter, in_place=True)
        torch.cuda.synchronize()
        assert res2.data_ptr() == d.data_ptr() and torch.equal(res2, res) and torch.equal(coef2, coef)


def test_single_outputs_of_the_staged_kernel():
    """Coefficients only (no residual pass) and residuals only give the same values as both together."""
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    y, jit = _case(5, 43, 24, 44)
    with MatchedFilter(0) as mf:
        d = torch.from_numpy(y).cuda()
        coef, res = mf.background(d, jit, 1.0, 5)
        coef1 = torch.empty_like(coef)
        res1 = torch.empty_like(res)
        P.tno_mf_background(mf.ctx, d, jit, 1.0, 5, coef1, None)
        P.tno_mf_background(mf.ctx, d, jit, 1.0, 5, None, res1)
        torch.cuda.synchronize()
        assert torch.equal(coef1, coef) and torch.equal(res1, res)


def test_static_pointing_and_errors():
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    rng = np.random.default_rng(9)
    T, H, W = 30, 8, 12
    y = (7.0 + rng.standard_normal((T, H, W))).astype(np.float32)
    still = np.zeros((T, 2), np.float32)
    with MatchedFilter(0) as mf:
        coef, res = mf.background(torch.from_numpy(y).cuda(), still, 1e9, 0)
        torch.cuda.synchronize()
        c = coef.cpu().numpy()
        assert np.allclose(c[0], y.mean(axis=0), atol=1e-5) and np.all(c[1:] == 0)      # only B is identifiable
        assert np.allclose(res.cpu().numpy(), y - y.mean(axis=0), atol=1e-5)
        d = torch.from_numpy(y).cuda()
        for bad in ((0.0, 1), (float("nan"), 1), (1.0, -1)):
            with pytest.raises(P.TnoMfError):
                P.tno_mf_background(mf.ctx, d, still, bad[0], bad[1], None, d)
        with pytest.raises(P.TnoMfError):
            P.tno_mf_background(mf.ctx, d, still, 1.0, 1, None, None)
