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


# ---- the basis itself, against the paper (PAPER.md:L67 and Eq. 1) ---------------------------
def test_basis_columns_are_the_papers_theta_k_after_the_constant():
    """PAPER.md:L67 prints the basis: theta_t = (x_t, y_t), theta_t^k = (x_t, y_t, x_t^2, y_t^2, x_t y_t); Eq. 1
    (L75) adds the background B itself, the constant column.  Rows listed by hand, with jitters whose six
    entries are pairwise different, so that any two swapped columns, a dropped square or a wrong sign fail."""
    jit = np.array([[2.0, 3.0], [-0.5, 0.25], [0.0, 0.0], [1.5, -4.0]], dtype=np.float32)
    want = np.array([[1.0, 2.0, 3.0, 4.0, 9.0, 6.0],
                     [1.0, -0.5, 0.25, 0.25, 0.0625, -0.125],
                     [1.0, 0.0, 0.0, 0.0, 0.0, 0.0],
                     [1.0, 1.5, -4.0, 2.25, 16.0, -6.0]])
    got = oracle.background_basis(jit)
    assert got.dtype == np.float64 and got.shape == (4, 6)
    assert np.array_equal(got, want)
    for a in range(6):                       # the rows above do tell every pair of columns apart
        for b in range(a + 1, 6):
            assert not np.array_equal(want[:, a], want[:, b])


def test_basis_promotes_the_float32_jitter_exactly():
    """The ABI carries the jitter as float32; the basis is formed in float64 from those values (products of two
    float32 numbers are exact in float64), not from a float64 jitter and not in float32."""
    j64 = np.array([[0.1, -0.3]])
    x, y = float(np.float32(0.1)), float(np.float32(-0.3))
    got = oracle.background_basis(j64)
    assert np.array_equal(got[0], np.array([1.0, x, y, x * x, y * y, x * y]))
    assert got[0, 1] != 0.1 and got[0, 3] != float(np.float32(x * x))


def test_background_returns_the_coefficients_in_the_papers_order():
    """A noiseless model planted with a basis typed out here from PAPER.md:L67 (no call to background_basis) is
    recovered coefficient by coefficient: B first, then B_theta in the order (x, y, x^2, y^2, xy)."""
    rng = np.random.default_rng(11)
    T, H, W = 40, 3, 4
    jit = (0.4 * rng.standard_normal((T, 2))).astype(np.float32)
    x, y = jit[:, 0].astype(np.float64), jit[:, 1].astype(np.float64)
    B, Bx, By, Bxx, Byy, Bxy = (rng.standard_normal((H, W)) * s for s in (50, 5, 4, 3, 2, 1))
    data = (B[None] + Bx[None] * x[:, None, None] + By[None] * y[:, None, None]
            + Bxx[None] * (x * x)[:, None, None] + Byy[None] * (y * y)[:, None, None]
            + Bxy[None] * (x * y)[:, None, None])
    beta, res = oracle.background(data.astype(np.float32), jit, 1e9, 0)
    for got, want in zip(beta, (B, Bx, By, Bxx, Byy, Bxy)):
        assert np.allclose(got, want, atol=2e-4)
    assert np.abs(res).max() < 2e-4
