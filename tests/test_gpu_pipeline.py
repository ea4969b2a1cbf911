"""The chain of PAPER.md section 3 on the device, end to end on a synthetic stack: raw frames = smooth scattered light
that changes from frame to frame + a static star field that moves with the pointing jitter + noise + one faint
mover.  downsample -> scattered-light fit -> subtract -> per-pixel background fit -> matched-filter search with the
max over the bank -> local-sigma scores -> non-maximum suppression: the mover comes out as the first candidate, at its
pixel and trajectory, and it would not without the two background steps."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


def test_raw_frames_to_candidate():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    rng = np.random.default_rng(11)
    T, H, n, f = 80, 128, 4, 4
    N = H // f
    jit = (0.12 * rng.standard_normal((T, 2))).astype(np.float32)
    phi = oracle.background_basis(jit)
    # star field: a smooth-ish static image and its first derivatives as the jitter response (Eq. 1's Taylor terms)
    yy, xx = np.mgrid[0:H, 0:H]
    stars = np.zeros((H, H))
    for _ in range(40):
        cx, cy, a = rng.uniform(0, H), rng.uniform(0, H), rng.uniform(50, 400)
        stars += a * np.exp(-((xx - cx) ** 2 + (yy - cy) ** 2) / (2 * 1.2 ** 2))
    gy, gx = np.gradient(stars)
    gyy, _ = np.gradient(gy)
    gxy, gxx = np.gradient(gx)
    beta = np.stack([stars, -gx, -gy, 0.5 * gxx, 0.5 * gyy, gxy])
    S = 60.0 + 25.0 * np.cumsum(rng.standard_normal((T, n, n)), axis=0) / np.sqrt(T) * 3
    raw = oracle.upsample(S, H) + np.einsum("tk,kij->tij", phi, beta) + rng.standard_normal((T, H, H))
    raw = raw.astype(np.float32)
    trajs = np.array([[vx, vy, 0, 0] for vx in (0.10, 0.16, 0.22) for vy in (-0.06, 0.0, 0.06)], np.float32)
    oracle.inject(raw, trajs[5:6], [70], [50], [1.6], 1.0, T / 2.0)           # peak 1.6 sigma per frame
    sigma = np.ones(T, np.float32)

    def detect(mf, frames):
        mx, ak, _, _ = mf.search_max(frames, sigma, trajs, 1.0, T / 2.0)
        _, _, z, _ = mf.best(mx[None].contiguous(), 63)
        _, top = mf.peaks(z, 4, ak)
        torch.cuda.synchronize()
        return mf.candidates_to_numpy(top[None])[0]

    with MatchedFilter(0, 5, 5.0) as mf:
        d = torch.from_numpy(raw).cuda()
        low = torch.empty((T, N, N), device="cuda")
        P.tno_mf_downsample(mf.ctx, d, f, low)
        b = torch.zeros((6, N, N), device="cuda")
        s = torch.zeros((T, n, n), device="cuda")
        loss, iters, _ = P.tno_mf_scatter_fit(mf.ctx, low, jit, 3.0, 500, 0.0, b, s)
        assert iters > 5
        clean = d.clone()
        P.tno_mf_scatter_subtract(mf.ctx, clean, s)
        coef, resid = mf.background(clean, jit, 3.0, 8, in_place=True)
        torch.cuda.synchronize()
        # the residual stack is noise-like: the stars (hundreds of sigma) and the scattered light (tens) are gone
        r = resid.cpu().numpy()
        assert abs(np.median(r)) < 0.2 and 0.8 < np.std(r) < 1.3
        c = detect(mf, resid)
        assert int(c["x"][0]) in (69, 70, 71) and int(c["y"][0]) in (49, 50, 51) and int(c["k"][0]) == 5
        assert c["snr"][0] > 8.0
        # without the background steps the same search finds stars, not the mover
        c_raw = detect(mf, d)
        assert not (abs(int(c_raw["x"][0]) - 70) <= 1 and abs(int(c_raw["y"][0]) - 50) <= 1)
