"""Pins for the oracle of the high-resolution background model (section 3.1: per-pixel regression on
the jitter basis with the Huber loss, solved by repeated least squares with clipped residuals)."""
import numpy as np
import pytest
import scipy.optimize

import oracle


def _case(seed, T=60, H=5, W=7, outliers=True):
    rng = np.random.default_rng(seed)
    jit = (0.4 * rng.standard_normal((T, 2))).astype(np.float32)
    phi = oracle.background_basis(jit)
    beta = rng.standard_normal((6, H, W)) * np.array([50, 5, 5, 2, 2, 2])[:, None, None]
    y = np.einsum("tk,khw->thw", phi, beta) + 0.5 * rng.standard_normal((T, H, W))
    if outliers:
        hit = rng.uniform(size=y.shape) < 0.05
        y = y + hit * rng.laplace(0, 20, size=y.shape)
    return y.astype(np.float32), jit, beta


def test_huge_delta_is_ordinary_least_squares():
    y, jit, _ = _case(1)
    beta, res = oracle.background(y, jit, 1e9, 3)
    phi = oracle.background_basis(jit)
    ref = np.linalg.lstsq(phi, y.astype(np.float64).reshape(60, -1), rcond=None)[0].reshape(6, 5, 7)
    assert np.allclose(beta, ref, rtol=1e-9, atol=1e-9)
    assert np.allclose(np.einsum("tk,thw->khw", phi, res), 0, atol=1e-8)        # normal equations


def test_fixed_point_is_the_huber_m_estimate():
    """After many iterations the estimating equation Phi^T psi_delta(r) = 0 holds, and the coefficients are
    those of a direct minimisation of the Huber loss (scipy, one pixel)."""
    y, jit, _ = _case(2)
    delta = 1.0
    beta, res = oracle.background(y, jit, delta, 400)
    phi = oracle.background_basis(jit)
    g = np.einsum("tk,thw->khw", phi, np.clip(res, -delta, delta))
    assert np.abs(g).max() < 1e-6
    yy = y[:, 2, 3].astype(np.float64)

    def huber(b):
        r = yy - phi @ b
        a = np.abs(r)
        return np.sum(np.where(a <= delta, 0.5 * r * r, delta * (a - 0.5 * delta)))
    opt = scipy.optimize.minimize(huber, beta[:, 2, 3] + 0.1, method="BFGS", options={"gtol": 1e-10})
    assert huber(beta[:, 2, 3]) <= opt.fun + 1e-8
    assert np.allclose(opt.x, beta[:, 2, 3], atol=2e-3)


def test_loss_decreases_and_outliers_are_resisted():
    y, jit, truth = _case(3)
    phi = oracle.background_basis(jit)

    def loss(beta, delta=1.0):
        r = y.astype(np.float64) - np.einsum("tk,khw->thw", phi, beta)
        a = np.abs(r)
        return np.sum(np.where(a <= delta, 0.5 * r * r, delta * (a - 0.5 * delta)))
    prev = None
    for n in (0, 1, 2, 5, 20):
        b, _ = oracle.background(y, jit, 1.0, n)
        cur = loss(b)
        assert prev is None or cur <= prev + 1e-9
        prev = cur
    ols, _ = oracle.background(y, jit, 1e9, 0)
    rob, _ = oracle.background(y, jit, 1.0, 50)
    assert np.abs(rob[0] - truth[0]).mean() < 0.6 * np.abs(ols[0] - truth[0]).mean()


def test_noiseless_model_is_recovered_exactly_and_static_pointing_degenerates_gracefully():
    rng = np.random.default_rng(4)
    jit = (0.4 * rng.standard_normal((30, 2))).astype(np.float32)
    phi = oracle.background_basis(jit)
    truth = rng.standard_normal((6, 3, 4))
    y = np.einsum("tk,khw->thw", phi, truth).astype(np.float32)
    beta, res = oracle.background(y, jit, 0.5, 10)
    assert np.allclose(beta, truth, atol=1e-5) and np.abs(res).max() < 1e-5
    still = np.zeros((30, 2), np.float32)                      # no jitter: only the constant is identifiable
    y2 = (7.0 + rng.standard_normal((30, 3, 4))).astype(np.float32)
    beta2, res2 = oracle.background(y2, still, 1e9, 0)
    assert np.allclose(beta2[0], y2.astype(np.float64).mean(axis=0)) and np.allclose(beta2[1:], 0)
    assert np.allclose(res2, y2 - y2.astype(np.float64).mean(axis=0))
