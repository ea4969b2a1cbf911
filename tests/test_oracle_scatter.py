"""Pins for the oracle of the low-resolution scattered-light model (section 3.1, Eq. 1-4): the bilinear
upsampling against torch's, the gradient against central differences, convexity facts, and the fit on data that
the model can represent exactly."""
import numpy as np
import torch

import oracle


def test_upsample_equals_torch_bilinear_and_is_a_partition_of_unity():
    rng = np.random.default_rng(0)
    for n, N in ((4, 32), (8, 24), (5, 5), (16, 128)):
        S = rng.standard_normal((3, n, n))
        ref = torch.nn.functional.interpolate(torch.from_numpy(S)[None], size=(N, N), mode="bilinear",
                                              align_corners=False)[0].numpy()
        assert np.allclose(oracle.upsample(S, N), ref, rtol=0, atol=1e-12)
        A = oracle.bilinear_matrix(N, n)
        assert np.allclose(A.sum(axis=1), 1.0) and np.all(A >= 0) and np.all((A > 0).sum(axis=1) <= 2)
    # a plane is reproduced away from the clamped border
    yy, xx = np.mgrid[0:8, 0:8]
    up = oracle.upsample(2.0 * xx + 3.0 * yy, 64)
    u = (np.arange(64) + 0.5) / 8 - 0.5
    assert np.allclose(up[8:56, 8:56], (2.0 * u[None, :] + 3.0 * u[:, None])[8:56, 8:56])


def test_huber_and_block_mean():
    a = np.array([-3.0, -1.0, 0.0, 0.5, 1.0, 2.0])
    assert np.allclose(oracle.huber(a, 1.0), [2.5, 0.5, 0.0, 0.125, 0.5, 1.5])      # Eq. 4, continuous at delta
    f = np.arange(2 * 4 * 6, dtype=np.float64).reshape(2, 4, 6)
    d = oracle.downsample(f, 2)
    assert d.shape == (2, 2, 3) and d[0, 0, 0] == (0 + 1 + 6 + 7) / 4 and d[1, 1, 2] == f[1, 2:4, 4:6].mean()


def _problem(seed, T=7, N=12, n=3, noise=0.3):
    rng = np.random.default_rng(seed)
    jit = (0.3 * rng.standard_normal((T, 2))).astype(np.float32)
    beta = rng.standard_normal((6, N, N)) * np.array([20, 3, 3, 1, 1, 1])[:, None, None]
    S = 5.0 * rng.standard_normal((T, n, n))
    phi = oracle.background_basis(jit)
    D = oracle.upsample(S, N) + np.einsum("tk,kij->tij", phi, beta) + noise * rng.standard_normal((T, N, N))
    return D, jit, beta, S


def test_gradient_against_central_differences():
    D, jit, beta, S = _problem(1)
    rng = np.random.default_rng(2)
    b0 = beta + 0.7 * rng.standard_normal(beta.shape)            # residuals on both branches of the loss
    S0 = S + 0.7 * rng.standard_normal(S.shape)
    delta = 0.5
    L, gb, gs = oracle.scatter_loss_grad(D, jit, delta, b0, S0)
    r = D - (oracle.upsample(S0, 12) + np.einsum("tk,kij->tij", oracle.background_basis(jit), b0))
    assert 0.2 < np.mean(np.abs(r) > delta) < 0.9
    h = 1e-6
    for idx in ((0, 3, 4), (2, 0, 11), (5, 7, 7)):
        e = np.zeros_like(b0); e[idx] = h
        num = (oracle.scatter_loss_grad(D, jit, delta, b0 + e, S0)[0] -
               oracle.scatter_loss_grad(D, jit, delta, b0 - e, S0)[0]) / (2 * h)
        assert abs(num - gb[idx]) < 1e-5 * max(1.0, abs(num))
    for idx in ((0, 0, 0), (3, 1, 2), (6, 2, 1)):
        e = np.zeros_like(S0); e[idx] = h
        num = (oracle.scatter_loss_grad(D, jit, delta, b0, S0 + e)[0] -
               oracle.scatter_loss_grad(D, jit, delta, b0, S0 - e)[0]) / (2 * h)
        assert abs(num - gs[idx]) < 1e-5 * max(1.0, abs(num))


def test_planted_model_is_a_stationary_point_and_the_fit_finds_its_prediction():
    D, jit, beta, S = _problem(3, noise=0.0)
    L, gb, gs = oracle.scatter_loss_grad(D, jit, 1.0, beta, S)
    assert L < 1e-18 and np.abs(gb).max() < 1e-9 and np.abs(gs).max() < 1e-9
    fb, fS, loss = oracle.scatter_fit(D, jit, 1.0, 3, max_iter=3000)
    assert loss < 1e-6
    pred = oracle.upsample(fS, 12) + np.einsum("tk,kij->tij", oracle.background_basis(jit), fb)
    assert np.abs(pred - D).max() < 5e-3
    # with noise and outliers the loss at the fit is below the loss at the planted parameters (it is the minimum)
    Dn, jit, beta, S = _problem(4, noise=0.3)
    Dn[2, 5, 5] += 40.0
    _, _, loss = oracle.scatter_fit(Dn, jit, 0.6, 3, max_iter=3000)
    assert loss <= oracle.scatter_loss_grad(Dn, jit, 0.6, beta, S)[0] + 1e-9
