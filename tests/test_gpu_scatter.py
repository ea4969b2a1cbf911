"""GPU parity of the low-resolution scattered-light model (section 3.1, Eq. 1-4) against the oracle, through
the C ABI: block-mean downsampling, loss and gradient, the L-BFGS fit (loss and prediction of the minimiser), and
the subtraction of the upsampled scattered light."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


from helpers import scatter_problem as _problem  # noqa: E402


@pytest.mark.parametrize("T,N,n", [(9, 24, 3), (5, 64, 8), (17, 40, 5), (3, 16, 16), (6, 33, 4),
                                   (2, 1040, 13),           # N > 1024: the gather form of the S gradient
                                   (11, 36, 4), (3, 512, 64),     # staged kernel: ragged last block, T % 8 != 0; paper size
                                   (19, 512, 64), (9, 512, 32),   # fused kernel (N = 512): several stages, ratio 8 and 16
                                   (8, 512, 96),                  # ... and a non-integer N / n
                                   (5, 256, 16), (4, 320, 8)])    # wide stencils (N / n = 16, 40) on the two-kernel path
def test_loss_and_gradient_match_oracle(T, N, n):
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    D, jit, beta, S = _problem(T + N + n, T, N, n)
    rng = np.random.default_rng(1)
    b0 = (beta + rng.standard_normal(beta.shape)).astype(np.float32)
    S0 = (S + rng.standard_normal(S.shape)).astype(np.float32)
    delta = 0.8
    L, gb, gs = oracle.scatter_loss_grad(D, jit, delta, b0, S0)
    with MatchedFilter(0) as mf:
        d = [torch.from_numpy(a).cuda() for a in (D, b0, S0)]
        ggb, ggs = torch.empty_like(d[1]), torch.empty_like(d[2])
        loss = P.tno_mf_scatter_lossgrad(mf.ctx, d[0], jit, delta, d[1], d[2], ggb, ggs)
        torch.cuda.synchronize()
    assert abs(loss - L) <= 2e-5 * L
    # float32 sums of up to T (beta) and (2N/n)^2 (S) terms of size <= delta * weight
    assert np.abs(ggb.cpu().numpy() - gb).max() <= 2e-5 * max(1.0, np.abs(gb).max())
    assert np.abs(ggs.cpu().numpy() - gs).max() <= 2e-5 * max(1.0, np.abs(gs).max())


def test_gradient_does_not_depend_on_what_earlier_kernels_left_on_chip():
    """The fused evaluation once multiplied a never-written pad element of its shared staging rows by a zero weight:
    NaN whenever an earlier kernel had left a NaN bit pattern there.  Repeated calls from fresh contexts, between
    kernels that fill shared memory with such patterns, must give the same finite gradient every time."""
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    T, N, n = 9, 512, 32
    D, jit, beta, S = _problem(T + N + n, T, N, n)
    rng = np.random.default_rng(1)
    b0 = (beta + rng.standard_normal(beta.shape)).astype(np.float32)
    S0 = (S + rng.standard_normal(S.shape)).astype(np.float32)
    ref = None
    for rep in range(12):
        # a sort of all-ones int32 keys goes through shared memory: 0xffffffff is a NaN when read as a float
        torch.sort(torch.full((1 << 16,), -1, dtype=torch.int32, device="cuda"))
        with MatchedFilter(0) as mf:
            d = [torch.from_numpy(a).cuda() for a in (D, b0, S0)]
            ggb, ggs = torch.full_like(d[1], float("nan")), torch.full_like(d[2], float("nan"))
            loss = P.tno_mf_scatter_lossgrad(mf.ctx, d[0], jit, 0.8, d[1], d[2], ggb, ggs)
            torch.cuda.synchronize()
        a, b = ggb.cpu().numpy(), ggs.cpu().numpy()
        assert np.isfinite(loss) and np.all(np.isfinite(a)) and np.all(np.isfinite(b)), rep
        if ref is None:
            ref = (loss, a, b)
        else:
            assert loss == ref[0] and np.array_equal(a, ref[1]) and np.array_equal(b, ref[2]), rep


def test_downsample_and_subtract():
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    rng = np.random.default_rng(2)
    f = (100.0 + rng.standard_normal((5, 48, 64))).astype(np.float32)
    with MatchedFilter(0) as mf:
        d = torch.from_numpy(f).cuda()
        out = torch.empty((5, 12, 16), device="cuda")
        P.tno_mf_downsample(mf.ctx, d, 4, out)
        torch.cuda.synchronize()
        assert np.abs(out.cpu().numpy() - oracle.downsample(f, 4)).max() <= 1e-5
        for side in (64, 45):                                        # 16-byte path and the scalar path
            sq = (100.0 + rng.standard_normal((4, side, side))).astype(np.float32)
            S = (10.0 * rng.standard_normal((4, 8, 8))).astype(np.float32)
            dsq = torch.from_numpy(sq).cuda()
            P.tno_mf_scatter_subtract(mf.ctx, dsq, torch.from_numpy(S).cuda())
            torch.cuda.synchronize()
            assert np.abs(dsq.cpu().numpy() - (sq - oracle.upsample(S, side))).max() <= 2e-5
        with pytest.raises(P.TnoMfError):
            P.tno_mf_downsample(mf.ctx, d, 5, torch.empty((5, 9, 12), device="cuda"))      # 5 does not divide 48


def test_fit_reaches_the_oracles_minimum():
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    T, N, n = 40, 32, 4
    D, jit, beta, S = _problem(7, T, N, n)
    delta = 1.0
    ob, oS, oL = oracle.scatter_fit(D, jit, delta, n, max_iter=2000)
    with MatchedFilter(0) as mf:
        d = torch.from_numpy(D).cuda()
        b = torch.zeros((6, N, N), device="cuda")
        s = torch.zeros((T, n, n), device="cuda")
        loss, iters, evals = P.tno_mf_scatter_fit(mf.ctx, d, jit, delta, 2000, 0.0, b, s)
        assert mf.stats()[0] > 3 * evals
        # the reported loss is the loss of the returned parameters
        gb, gs = torch.empty_like(b), torch.empty_like(s)
        again = P.tno_mf_scatter_lossgrad(mf.ctx, d, jit, delta, b, s, gb, gs)
        torch.cuda.synchronize()
        # reproducible: the same call gives the same bits
        b2 = torch.zeros_like(b)
        s2 = torch.zeros_like(s)
        loss2, iters2, _ = P.tno_mf_scatter_fit(mf.ctx, d, jit, delta, 2000, 0.0, b2, s2)
        assert loss2 == loss and iters2 == iters and torch.equal(b2, b) and torch.equal(s2, s)
    assert abs(again - loss) <= 1e-6 * loss
    start = oracle.scatter_loss_grad(D, jit, delta, np.zeros_like(beta), np.zeros_like(S))[0]
    assert loss < 0.05 * start and 0 < iters <= 2000
    assert abs(loss - oL) <= 1e-4 * oL, (loss, oL, iters, evals)         # the convex minimum, to float32 resolution
    pred_g = oracle.upsample(s.cpu().numpy(), N) + np.einsum("tk,kij->tij", oracle.background_basis(jit),
                                                             b.cpu().numpy().astype(np.float64))
    pred_o = oracle.upsample(oS, N) + np.einsum("tk,kij->tij", oracle.background_basis(jit), ob)
    assert np.sqrt(np.mean((pred_g - pred_o) ** 2)) < 0.02           # noise is 0.3: the fits agree far below it


def test_fit_parity_on_a_longer_stack():
    """The fit at 200 frames of 128 x 128 (n = 16): the convex minimum and the prediction of scipy's L-BFGS-B (the
    oracle; its result is stored by tests/golden/make_scatter_golden.py, which takes the oracle a quarter of an hour)
    are reached from zeros, and two calls give the same bits."""
    torch = _torch()
    import os
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    T, N, n = 200, 128, 16
    D, jit, beta, S = _problem(21, T, N, n)
    delta = 1.0
    gold = np.loadtxt(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "scatter_fit_T200_N128_n16.txt"))
    oL, samples = gold[0, 3], gold[1:]
    with MatchedFilter(0) as mf:
        d = torch.from_numpy(D).cuda()
        b = torch.zeros((6, N, N), device="cuda")
        s = torch.zeros((T, n, n), device="cuda")
        loss, iters, evals = P.tno_mf_scatter_fit(mf.ctx, d, jit, delta, 3000, 0.0, b, s)
        b2, s2 = torch.zeros_like(b), torch.zeros_like(s)
        loss2, iters2, _ = P.tno_mf_scatter_fit(mf.ctx, d, jit, delta, 3000, 0.0, b2, s2)
        assert loss2 == loss and iters2 == iters and torch.equal(b2, b) and torch.equal(s2, s)
    assert abs(loss - oL) <= 2e-4 * oL, (loss, oL, iters, evals)
    basis = oracle.background_basis(jit)
    pred_g = oracle.upsample(s.cpu().numpy(), N) + np.einsum("tk,kij->tij", basis, b.cpu().numpy().astype(np.float64))
    t, i, j = samples[:, 0].astype(int), samples[:, 1].astype(int), samples[:, 2].astype(int)
    assert np.sqrt(np.mean((pred_g[t, i, j] - samples[:, 3]) ** 2)) < 0.03      # noise is 0.3


def test_fit_on_exact_data_and_errors():
    torch = _torch()
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    T, N, n = 8, 24, 3
    D, jit, beta, S = _problem(9, T, N, n, noise=0.0, outliers=0.0)
    with MatchedFilter(0) as mf:
        d = torch.from_numpy(D).cuda()
        b = torch.zeros((6, N, N), device="cuda")
        s = torch.zeros((T, n, n), device="cuda")
        loss, iters, _ = P.tno_mf_scatter_fit(mf.ctx, d, jit, 1.0, 3000, 0.0, b, s)
        torch.cuda.synchronize()
        pred = oracle.upsample(s.cpu().numpy(), N) + np.einsum("tk,kij->tij", oracle.background_basis(jit),
                                                               b.cpu().numpy().astype(np.float64))
        assert np.abs(pred - D).max() < 0.05 and loss < 1e-3 * T * N * N
        for bad in ((0.0, 10, 0.0), (1.0, -1, 0.0), (1.0, 10, -1.0)):
            with pytest.raises(P.TnoMfError):
                P.tno_mf_scatter_fit(mf.ctx, d, jit, bad[0], bad[1], bad[2], b, s)
