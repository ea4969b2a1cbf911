"""CPU oracle (float64) for the matched-filter trajectory search -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2209_09848_b200``) never does, and this package never imports the product.

The arithmetic lives in ``tno_oracle.c`` (plain C, float64, one exp per tap in ``point``); this
file only marshals numpy arrays.  ``topk`` is the plain definition: threshold, then a library
sort by (SNR descending, y ascending, x ascending) -- BASELINE.json:north_star "per-trajectory
top-K candidate list above a threshold".

Pins: tests/test_oracle_pins.py.  No function here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
from typing import Optional, Tuple

import numpy as np

from .build import build as _build

_lib = ctypes.CDLL(_build())
_f32p = ctypes.POINTER(ctypes.c_float)
_f64p = ctypes.POINTER(ctypes.c_double)
_i32p = ctypes.POINTER(ctypes.c_int)

_lib.tno_oracle_threads.restype = ctypes.c_int
_lib.tno_oracle_point.restype = ctypes.c_int
_lib.tno_oracle_point.argtypes = [_f32p] + [ctypes.c_int] * 7 + [_f32p, _f32p, ctypes.c_float,
                                  ctypes.c_float, ctypes.c_int, ctypes.c_int, _f64p, _f64p, _f64p]
_lib.tno_oracle_map.restype = ctypes.c_int
_lib.tno_oracle_map.argtypes = [_f32p] + [ctypes.c_int] * 7 + [_f32p, _f32p, ctypes.c_int,
                                ctypes.c_float, ctypes.c_float] + [ctypes.c_int] * 4 + [_f64p] * 3
_lib.tno_oracle_inject.restype = ctypes.c_int
_lib.tno_oracle_inject.argtypes = [_f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _f32p, _i32p,
                                   _i32p, _f32p, ctypes.c_int, ctypes.c_float, ctypes.c_float]

CAND_DTYPE = np.dtype([("snr", np.float64), ("x", np.int32), ("y", np.int32), ("k", np.int32)])


_lib.tno_oracle_point_ex.restype = ctypes.c_int
_lib.tno_oracle_point_ex.argtypes = [_f32p] + [ctypes.c_int] * 7 + [_f32p, _f32p, _f32p, _f32p, ctypes.c_int, _f32p, ctypes.c_float,
                                     ctypes.c_float, ctypes.c_int, ctypes.c_int, _f64p, _f64p, _f64p]
_lib.tno_oracle_map_ex.restype = ctypes.c_int
_lib.tno_oracle_map_ex.argtypes = [_f32p] + [ctypes.c_int] * 7 + [_f32p, _f32p, _f32p, _f32p, ctypes.c_int, _f32p, ctypes.c_int,
                                   ctypes.c_float, ctypes.c_float] + [ctypes.c_int] * 4 + [_f64p] * 3
_lib.tno_oracle_inject_ex.restype = ctypes.c_int
_lib.tno_oracle_inject_ex.argtypes = [_f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _f32p, _f32p, _f32p,
                                      _i32p, _i32p, _f32p, ctypes.c_int, ctypes.c_float, ctypes.c_float]


_lib.tno_oracle_inject_mode.restype = ctypes.c_int
_lib.tno_oracle_inject_mode.argtypes = [_f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _f32p, _f32p, ctypes.c_int,
                                        _f32p, _i32p, _i32p, _f32p, ctypes.c_int, ctypes.c_float, ctypes.c_float]
_lib.tno_oracle_set_prf_table.restype = ctypes.c_int
_lib.tno_oracle_set_prf_table.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.c_int]
_lib.tno_oracle_set_prf_table2d.restype = ctypes.c_int
_lib.tno_oracle_set_prf_table2d.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_int]


def _opt(a, shape):
    """Optional float32 array -> (keep-alive array, pointer or None)."""
    if a is None:
        return None, None
    a = _f32(a, shape)
    return a, a.ctypes.data_as(_f32p)


def _valid_ptr(valid, frames):
    """Pointer to the validity weights (same shape as the frames buffer), or None."""
    if valid is None:
        return None
    assert valid.dtype == np.float32 and valid.flags.c_contiguous and valid.shape == frames.shape
    return valid.ctypes.data_as(_f32p)


_f64c = ctypes.POINTER(ctypes.c_double)


def _mode(shift_stack, filter, prf_table) -> int:
    """Filter mode of tap1 / tap2 in tno_oracle.c (0 point-sampled Gaussian, 1 shift-stack, 2 pixel-integrated
    Gaussian, 3 tabulated separable, 4 tabulated non-separable); mode 3 installs `prf_table` ([n_phase, 5]
    fractions) first, mode 4 the 2-D table ([n_phase_y, n_phase_x, 5, 5])."""
    mode = int(filter) if filter else int(bool(shift_stack))
    assert mode in (0, 1, 2, 3, 4)
    if mode == 3:
        tab = np.ascontiguousarray(prf_table, dtype=np.float64)
        assert tab.ndim == 2 and tab.shape[1] == 5 and tab.shape[0] >= 1
        rc = _lib.tno_oracle_set_prf_table(tab.ctypes.data_as(_f64c), int(tab.shape[0]))
        assert rc == 0
    if mode == 4:
        # non-separable tabulated PRF: [n_phase_y, n_phase_x, 5, 5], entry [ry, rx, j + 2, i + 2]
        tab = np.ascontiguousarray(prf_table, dtype=np.float64)
        assert tab.ndim == 4 and tab.shape[2:] == (5, 5) and tab.shape[0] >= 1 and tab.shape[1] >= 1
        rc = _lib.tno_oracle_set_prf_table2d(tab.ctypes.data_as(_f64c), int(tab.shape[0]), int(tab.shape[1]))
        assert rc == 0
    return mode


def threads() -> int:
    return int(_lib.tno_oracle_threads())


def _f32(a, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float32)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def _geom(frames: np.ndarray, window, full_shape):
    T, wh, ww = frames.shape
    if window is None:
        assert full_shape is None or tuple(full_shape) == (wh, ww)
        return T, wh, ww, 0, 0, ww, wh
    wx0, wy0 = window
    H, W = full_shape
    return T, H, W, int(wx0), int(wy0), ww, wh


def point(frames, sigma_t, traj, prf_sigma, t0, x, y, window=None, full_shape=None,
          times=None, jitter=None, valid=None, shift_stack: bool = False, filter: int = 0,
          prf_table=None) -> Tuple[float, float, float]:
    """(snr, N, D) at start pixel (x, y) for one trajectory (vx, vy, ax, ay).  times: frame times [T]
    (default the frame index), jitter: pointing offsets [T, 2] in px added to the track (default 0),
    valid: per-pixel weights of D with the layout of frames (default 1; N uses the frames as they are)."""
    frames = _f32(frames)
    T, H, W, wx0, wy0, ww, wh = _geom(frames, window, full_shape)
    sigma_t = _f32(sigma_t, (T,))
    traj = _f32(traj, (4,))
    N, D, S = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _ta, tp = _opt(times, (T,))
    _ja, jp = _opt(jitter, (T, 2))
    rc = _lib.tno_oracle_point_ex(frames.ctypes.data_as(_f32p), T, H, W, wx0, wy0, ww, wh,
                                  sigma_t.ctypes.data_as(_f32p), tp, jp, _valid_ptr(valid, frames),
                                  _mode(shift_stack, filter, prf_table), traj.ctypes.data_as(_f32p), float(prf_sigma),
                                  float(t0),
                                  int(x), int(y),
                                  ctypes.byref(N), ctypes.byref(D), ctypes.byref(S))
    if rc != 0:
        raise ValueError("oracle.point: tap outside the supplied window (rc=%d)" % rc)
    return S.value, N.value, D.value


def snr_map(frames, sigma_t, trajs, prf_sigma, t0, region=None, window=None, full_shape=None,
            return_ND: bool = False, times=None, jitter=None, valid=None, shift_stack: bool = False,
            filter: int = 0, prf_table=None):
    """float64 [K, h, w] SNR for start pixels x in [x_lo, x_hi), y in [y_lo, y_hi)
    (region = (x_lo, x_hi, y_lo, y_hi), default the whole frame)."""
    frames = _f32(frames)
    T, H, W, wx0, wy0, ww, wh = _geom(frames, window, full_shape)
    sigma_t = _f32(sigma_t, (T,))
    trajs = _f32(trajs)
    assert trajs.ndim == 2 and trajs.shape[1] == 4
    K = trajs.shape[0]
    x_lo, x_hi, y_lo, y_hi = (0, W, 0, H) if region is None else region
    out = np.empty((K, y_hi - y_lo, x_hi - x_lo), dtype=np.float64)
    oN = np.empty_like(out) if return_ND else None
    oD = np.empty_like(out) if return_ND else None
    _ta, tp = _opt(times, (T,))
    _ja, jp = _opt(jitter, (T, 2))
    rc = _lib.tno_oracle_map_ex(frames.ctypes.data_as(_f32p), T, H, W, wx0, wy0, ww, wh,
                             sigma_t.ctypes.data_as(_f32p), tp, jp, _valid_ptr(valid, frames),
                             _mode(shift_stack, filter, prf_table), trajs.ctypes.data_as(_f32p), K,
                             float(prf_sigma), float(t0), int(x_lo), int(x_hi), int(y_lo),
                             int(y_hi), out.ctypes.data_as(_f64p),
                             oN.ctypes.data_as(_f64p) if return_ND else None,
                             oD.ctypes.data_as(_f64p) if return_ND else None)
    if rc != 0:
        raise ValueError("oracle.snr_map failed (rc=%d): -1 = tap outside the window" % rc)
    return (out, oN, oD) if return_ND else out


def topk(snr: np.ndarray, ktop: int, threshold: float, k_index: int = 0,
         origin: Tuple[int, int] = (0, 0)) -> np.ndarray:
    """Candidates of ONE map [h, w]: all pixels with snr >= threshold, ordered by
    (snr descending, y ascending, x ascending), first `ktop` of them, padded to `ktop` records
    with (-inf, -1, -1, k)."""
    snr = np.asarray(snr, dtype=np.float64)
    ys, xs = np.nonzero(snr >= threshold)
    vals = snr[ys, xs]
    order = np.lexsort((xs, ys, -vals))[:ktop]     # last key is the primary one
    out = np.empty(ktop, dtype=CAND_DTYPE)
    out["snr"] = -np.inf
    out["x"] = -1
    out["y"] = -1
    out["k"] = k_index
    n = order.size
    out["snr"][:n] = vals[order]
    out["x"][:n] = xs[order] + origin[0]
    out["y"][:n] = ys[order] + origin[1]
    return out


def inject(frames: np.ndarray, trajs, xs, ys, amps, prf_sigma, t0, times=None, jitter=None, filter: int = 0,
           prf_table=None) -> None:
    """In place: add amp * g(p - c_t) for each source (full-frame float32 [T, H, W] buffer); g is the filter
    of mode `filter` (0: the point-sampled Gaussian)."""
    assert frames.dtype == np.float32 and frames.flags.c_contiguous and frames.ndim == 3
    T, H, W = frames.shape
    trajs = _f32(trajs)
    n = trajs.shape[0]
    xs = np.ascontiguousarray(xs, dtype=np.int32)
    ys = np.ascontiguousarray(ys, dtype=np.int32)
    amps = _f32(amps, (n,))
    assert xs.shape == (n,) and ys.shape == (n,) and trajs.shape == (n, 4)
    _ta, tp = _opt(times, (T,))
    _ja, jp = _opt(jitter, (T, 2))
    if filter:
        rc = _lib.tno_oracle_inject_mode(frames.ctypes.data_as(_f32p), T, H, W, tp, jp,
                                         ctypes.c_int(_mode(False, filter, prf_table)),
                                         trajs.ctypes.data_as(_f32p), xs.ctypes.data_as(_i32p),
                                         ys.ctypes.data_as(_i32p), amps.ctypes.data_as(_f32p), n,
                                         ctypes.c_float(prf_sigma), ctypes.c_float(t0))
    else:
        rc = _lib.tno_oracle_inject_ex(frames.ctypes.data_as(_f32p), T, H, W, tp, jp,
                                       trajs.ctypes.data_as(_f32p), xs.ctypes.data_as(_i32p),
                                       ys.ctypes.data_as(_i32p), amps.ctypes.data_as(_f32p), n,
                                       float(prf_sigma), float(t0))
    assert rc == 0


# ---- interpreting scores (section 3.3): max over the bank, local-sigma units ----------
_lib.tno_oracle_best.restype = ctypes.c_int
_lib.tno_oracle_best.argtypes = [_f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _f32p, _i32p]
for _name in ("tno_oracle_local_z", "tno_oracle_local_z_sep"):
    getattr(_lib, _name).restype = ctypes.c_int
    getattr(_lib, _name).argtypes = [_f32p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _f64p, _f64p]


def best(snr):
    """(max over trajectories float32 [H, W], argmax int32 [H, W], smallest k on ties) of float32
    maps [K, H, W]."""
    snr = _f32(snr)
    K, H, W = snr.shape
    m = np.empty((H, W), np.float32)
    a = np.empty((H, W), np.int32)
    rc = _lib.tno_oracle_best(snr.ctypes.data_as(_f32p), K, H, W, m.ctypes.data_as(_f32p),
                              a.ctypes.data_as(_i32p))
    if rc != 0:
        raise ValueError("tno_oracle_best failed (%d)" % rc)
    return m, a


def local_z(m, box: int = 255, literal: bool = False):
    """(Z = M / sigma_box float64 [H, W], sigma_box float64 [H, W]): scores in units of the standard
    deviation of the scores in the box x box square centred on each pixel, clipped to the frame
    (PAPER.md:L124).  literal=True evaluates the two-pass definition pixel by pixel (small maps)."""
    m = _f32(m)
    H, W = m.shape
    z = np.empty((H, W), np.float64)
    s = np.empty((H, W), np.float64)
    fn = _lib.tno_oracle_local_z if literal else _lib.tno_oracle_local_z_sep
    rc = fn(m.ctypes.data_as(_f32p), H, W, int(box), z.ctypes.data_as(_f64p), s.ctypes.data_as(_f64p))
    if rc != 0:
        raise ValueError("tno_oracle_local_z failed (%d)" % rc)
    return z, s


def peaks(score, radius: int, threshold: float = -np.inf):
    """Non-maximum suppression of a score map [H, W] ("so one object yields one candidate";
    DESIGN.md reading e6): pixel p is a peak iff score(p) >= threshold and, for every other pixel q of the frame
    with |qx - px| <= radius and |qy - py| <= radius, score(p) > score(q), or score(p) == score(q) and p comes
    first in row-major order.  Returns the boolean peak mask.  Written as the definition, one window offset at
    a time (numpy float64)."""
    z = np.asarray(score, dtype=np.float64)
    H, W = z.shape
    r = int(radius)
    keep = z >= threshold
    pad = np.full((H + 2 * r, W + 2 * r), -np.inf)
    pad[r:r + H, r:r + W] = z
    for dy in range(-r, r + 1):
        for dx in range(-r, r + 1):
            if dy == 0 and dx == 0:
                continue
            q = pad[r + dy:r + dy + H, r + dx:r + dx + W]          # score of the neighbour at offset (dx, dy)
            q_is_later = dy > 0 or (dy == 0 and dx > 0)
            keep &= (z > q) | ((z == q) & q_is_later)
    return keep


# ---- high-resolution background model (section 3.1) ---------------------------
def background_basis(jitter) -> np.ndarray:
    """[T, 6] float64 basis (1, x, y, x^2, y^2, x y) of the per-pixel model of PAPER.md Eq. 1: the background
    B plus its 2nd-order Taylor expansion B_theta in the pointing jitter theta_t = (x_t, y_t) (L66)."""
    j = np.asarray(jitter, dtype=np.float32).astype(np.float64)
    x, y = j[:, 0], j[:, 1]
    return np.stack([np.ones_like(x), x, y, x * x, y * y, x * y], axis=1)


def background(frames, jitter, delta: float, n_iter: int):
    """Per-pixel robust fit of the background model with the scattered light already removed:
        y_t(p) = B(p) + B_theta(p) . theta_t^k + eps,   minimise sum_t L_delta(residual)   (Eq. 2-4)
    by "repeated least squares solves, alternated with clipping the residuals (Huber 1977)", every pixel
    regressed "against the same input data", so one pseudo-inverse serves all (L98-100):
        beta_0 = pinv(Phi) y ;   beta_{i+1} = beta_i + pinv(Phi) clip(y - Phi beta_i, -delta, +delta).
    Returns (coefficients float64 [6, H, W], residual stack float64 [T, H, W])."""
    y = np.asarray(frames, dtype=np.float32).astype(np.float64)
    T, H, W = y.shape
    phi = background_basis(jitter)
    pinv = np.linalg.pinv(phi)                       # [6, T]
    Y = y.reshape(T, H * W)
    beta = pinv @ Y
    d = float(np.float32(delta))
    for _ in range(int(n_iter)):
        r = Y - phi @ beta
        beta = beta + pinv @ np.clip(r, -d, d)
    r = Y - phi @ beta
    return beta.reshape(6, H, W), r.reshape(T, H, W)


# ---- low-resolution scattered-light model (section 3.1, Eq. 1-4) ------------------------------
def bilinear_matrix(n_out: int, n_in: int) -> np.ndarray:
    """[n_out, n_in] matrix of 1-D bilinear upsampling (reading s2): output pixel i has its centre at
    u = (i + 1/2) n_in / n_out - 1/2 in input pixel units, clamped to [0, n_in - 1]; it is the weighted
    combination of the two nearest input pixels, floor(u) with weight 1 - frac(u) and floor(u) + 1 (clamped) with
    weight frac(u) -- "the high resolution pixel is weighted combination of the 4 nearest low resolution points"
     in two dimensions."""
    A = np.zeros((n_out, n_in))
    for i in range(n_out):
        u = min(max((i + 0.5) * n_in / n_out - 0.5, 0.0), n_in - 1.0)
        i0 = int(np.floor(u))
        i1 = min(i0 + 1, n_in - 1)
        w = u - i0
        A[i, i0] += 1.0 - w
        A[i, i1] += w
    return A


def upsample(S, N: int) -> np.ndarray:
    """U(S): [..., n, n] -> [..., N, N], bilinear in both axes (Eq. 1)."""
    S = np.asarray(S, dtype=np.float64)
    A = bilinear_matrix(N, S.shape[-1])
    return np.einsum("ia,...ab,jb->...ij", A, S, A)


def huber(a, delta):
    """Eq. 4 with the lost bar restored: a^2 / 2 for |a| <= delta, delta (|a| - delta / 2) otherwise."""
    a = np.abs(a)
    return np.where(a <= delta, 0.5 * a * a, delta * (a - 0.5 * delta))


def scatter_loss_grad(D, jitter_xy, delta, beta, S):
    """Loss of Eq. 2-3 and its gradient for the low-resolution model of Eq. 1,
         pred_t = U(S_t) + sum_k phi_k(theta_t) beta_k,   L = sum_{t,i,j} L_delta(D_t - pred_t),
    phi = (1, x, y, x^2, y^2, x y) (background_basis), beta [6, N, N], S [T, n, n].
    Returns (L, dL/dbeta [6, N, N], dL/dS [T, n, n]) in float64: dL/dpred = -clip(r, -delta, delta), pushed
    through the transposes of the two linear maps."""
    D = np.asarray(D, dtype=np.float64)
    T, N, _ = D.shape
    phi = background_basis(jitter_xy)
    beta = np.asarray(beta, dtype=np.float64)
    S = np.asarray(S, dtype=np.float64)
    r = D - (upsample(S, N) + np.einsum("tk,kij->tij", phi, beta))
    L = float(huber(r, delta).sum())
    psi = np.clip(r, -delta, delta)
    A = bilinear_matrix(N, S.shape[-1])
    g_beta = -np.einsum("tk,tij->kij", phi, psi)
    g_S = -np.einsum("ia,tij,jb->tab", A, psi, A)
    return L, g_beta, g_S


def scatter_fit(D, jitter_xy, delta, n: int, max_iter: int = 500, gtol: float = 1e-8):
    """Minimise the loss over (beta, S) with L-BFGS from zero ("We minimize this convex loss over
    B, B_theta, S_t using the L-BFGS (Zhu et al. 1995) algorithm"): scipy's L-BFGS-B, the implementation of that
    paper, serves as the step.  Returns (beta, S, loss).  The split of a time-constant smooth component between S
    and B is not determined by the loss; the prediction and the loss are."""
    import scipy.optimize
    D = np.asarray(D, dtype=np.float64)
    T, N, _ = D.shape
    nb = 6 * N * N

    def fun(x):
        L, gb, gs = scatter_loss_grad(D, jitter_xy, delta, x[:nb].reshape(6, N, N), x[nb:].reshape(T, n, n))
        return L, np.concatenate([gb.ravel(), gs.ravel()])
    res = scipy.optimize.minimize(fun, np.zeros(nb + T * n * n), jac=True, method="L-BFGS-B",
                                  options={"maxiter": max_iter, "gtol": gtol, "ftol": 0.0, "maxcor": 10,
                                           "maxfun": 10 * max_iter})
    return res.x[:nb].reshape(6, N, N), res.x[nb:].reshape(T, n, n), float(res.fun)


def downsample(frames, f: int) -> np.ndarray:
    """Mean over f x f blocks: "the data downsampled to 512 x 512 from 2048 x 2048" (reading s1)."""
    a = np.asarray(frames, dtype=np.float64)
    T, H, W = a.shape
    return a.reshape(T, H // f, f, W // f, f).mean(axis=(2, 4))
