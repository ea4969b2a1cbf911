"""Out-of-bounds writes would be silent in the parity tests if they landed in unused memory: here every output of
the calls added after the search (background, scattered-light model, peaks, fused max, flux) lives inside a larger
buffer whose margins hold a bit pattern, and the margins must come back untouched -- also for ragged sizes that end
in the middle of a block."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

PAD = 4096            # floats on each side (16 KB: keeps the 16-byte alignment the fast kernels look for)
MAGIC = -1.2345678e30


class Guarded:
    def __init__(self, torch, shape, dtype=None):
        dtype = dtype or torch.float32
        n = int(np.prod(shape))
        self.buf = torch.full((n + 2 * PAD,), MAGIC if dtype == torch.float32 else -1234567, dtype=dtype, device="cuda")
        self.t = self.buf[PAD:PAD + n].view(*shape)
        self.fill = self.buf[0].clone()

    def intact(self):
        return bool((self.buf[:PAD] == self.fill).all()) and bool((self.buf[-PAD:] == self.fill).all())


@pytest.mark.parametrize("T,H,W", [(19, 36, 52), (10, 33, 47), (9, 64, 64), (3, 4, 132)])
def test_margins_survive(T, H, W):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    rng = np.random.default_rng(T + H + W)
    jit = (0.2 * rng.standard_normal((T, 2))).astype(np.float32)
    sigma = np.ones(T, np.float32)
    trajs = np.array([[0.1, -0.2, 0, 0], [0.1, 0.15, 0, 0.001], [-0.3, 0.05, 0, 0]], np.float32)
    with MatchedFilter(0, 4, 1.0) as mf:
        frames = Guarded(torch, (T, H, W))
        frames.t.copy_(torch.from_numpy(rng.standard_normal((T, H, W)).astype(np.float32)))
        # background: coefficients and residuals, out of place and in place
        coef, resid = Guarded(torch, (6, H, W)), Guarded(torch, (T, H, W))
        P.tno_mf_background(mf.ctx, frames.t, jit, 1.0, 3, coef.t, resid.t)
        P.tno_mf_background(mf.ctx, frames.t, jit, 1.0, 2, coef.t, frames.t)
        # fused max, maps, lists
        mx, ak = Guarded(torch, (H, W)), Guarded(torch, (H, W), torch.int32)
        maps, top = Guarded(torch, (3, H, W)), Guarded(torch, (3, 4, 4), torch.int32)
        P.tno_mf_search_max(mf.ctx, frames.t, None, sigma, None, jit, trajs, 1.0, T / 2.0, mx.t, ak.t, maps.t, top.t)
        flux = Guarded(torch, (3, H, W))
        P.tno_mf_flux(mf.ctx, maps.t, flux.t)
        # scores and peaks
        m2, a2, z = Guarded(torch, (H, W)), Guarded(torch, (H, W), torch.int32), Guarded(torch, (H, W))
        t2 = Guarded(torch, (4, 4), torch.int32)
        P.tno_mf_best(mf.ctx, maps.t, 9, m2.t, a2.t, z.t, t2.t)
        pk, t3 = Guarded(torch, (H, W)), Guarded(torch, (4, 4), torch.int32)
        P.tno_mf_peaks(mf.ctx, z.t, a2.t, 3, pk.t, t3.t)
        torch.cuda.synchronize()
        for g in (frames, coef, resid, mx, ak, maps, top, flux, m2, a2, z, t2, pk, t3):
            assert g.intact()
        # scattered-light model on a square low-resolution version of the stack
        if H % 4 == 0 and W % 4 == 0:
            N, n = 32, 4
            low_src = Guarded(torch, (T, 4 * N, 4 * N))
            low_src.t.copy_(torch.from_numpy(rng.standard_normal((T, 4 * N, 4 * N)).astype(np.float32)))
            low = Guarded(torch, (T, N, N))
            P.tno_mf_downsample(mf.ctx, low_src.t, 4, low.t)
            beta, S = Guarded(torch, (6, N, N)), Guarded(torch, (T, n, n))
            beta.t.zero_()
            S.t.zero_()
            gb, gs = Guarded(torch, (6, N, N)), Guarded(torch, (T, n, n))
            P.tno_mf_scatter_lossgrad(mf.ctx, low.t, jit, 1.0, beta.t, S.t, gb.t, gs.t)
            P.tno_mf_scatter_fit(mf.ctx, low.t, jit, 1.0, 20, 0.0, beta.t, S.t)
            P.tno_mf_scatter_subtract(mf.ctx, low_src.t, S.t)
            torch.cuda.synchronize()
            for g in (low_src, low, beta, S, gb, gs):
                assert g.intact()
