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


def _all_outputs(torch, P, MatchedFilter, fill_byte, T, H, W, force_generic):
    """Every output-only buffer of the calls below starts as `fill_byte` bytes (0x00: zeros; 0xff: NaN as floats, -1 as
    integers); returns the outputs as numpy arrays."""
    rng = np.random.default_rng(T + H + W)
    jit = (0.2 * rng.standard_normal((T, 2))).astype(np.float32)
    sigma = np.ones(T, np.float32)
    trajs = np.array([[0.1, -0.2, 0, 0], [0.1, 0.2, 0, 0], [0.1, 0.15, 0, 0.001], [-0.3, 0.05, 0, 0]], np.float32)
    frames = torch.from_numpy(rng.standard_normal((T, H, W)).astype(np.float32)).cuda()
    valid = torch.from_numpy((rng.random((T, H, W)) > 0.05).astype(np.float32)).cuda()

    def out(shape, dtype=torch.float32):
        n = int(np.prod(shape)) * (4 if dtype in (torch.float32, torch.int32) else 1)
        raw = torch.full((n,), fill_byte, dtype=torch.uint8, device="cuda")
        return raw.view(dtype).view(*shape)

    res = {}
    with MatchedFilter(0, 4, 1.0, force_generic=force_generic) as mf:
        coef, resid = out((6, H, W)), out((T, H, W))
        P.tno_mf_background(mf.ctx, frames, jit, 1.0, 3, coef, resid)
        maps, top = out((4, H, W)), out((4, 4, 4), torch.int32)
        P.tno_mf_search(mf.ctx, frames, sigma, trajs, 1.0, T / 2.0, maps, top)
        mmaps, mtop = out((4, H, W)), out((4, 4, 4), torch.int32)
        P.tno_mf_search_masked(mf.ctx, frames, valid, sigma, None, jit, trajs, 1.0, T / 2.0, mmaps, mtop)
        mx, ak = out((H, W)), out((H, W), torch.int32)
        xmaps, xtop = out((4, H, W)), out((4, 4, 4), torch.int32)
        P.tno_mf_search_max(mf.ctx, frames, None, sigma, None, None, trajs, 1.0, T / 2.0, mx, ak, xmaps, xtop)
        flux = out((4, H, W))
        P.tno_mf_flux(mf.ctx, xmaps, flux)
        m2, a2, z, t2 = out((H, W)), out((H, W), torch.int32), out((H, W)), out((4, 4), torch.int32)
        P.tno_mf_best(mf.ctx, maps, 9, m2, a2, z, t2)
        zs = out((H, W))
        P.tno_mf_local_z_static(mf.ctx, m2, 9, zs)
        pk, t3 = out((H, W)), out((4, 4), torch.int32)
        P.tno_mf_peaks(mf.ctx, z, a2, 3, pk, t3)
        torch.cuda.synchronize()
        for name, t in (("coef", coef), ("resid", resid), ("maps", maps), ("top", top), ("mmaps", mmaps), ("mtop", mtop),
                        ("mx", mx), ("ak", ak), ("xmaps", xmaps), ("xtop", xtop), ("flux", flux), ("m2", m2), ("a2", a2),
                        ("z", z), ("t2", t2), ("zs", zs), ("pk", pk), ("t3", t3)):
            res[name] = t.cpu().numpy().view(np.uint32).copy()
        # the scattered-light calls on a square stack: N = 512 takes the fused evaluation, N = 32 the two-kernel one
        for N, n in ((512, 32), (32, 4)):
            src = torch.from_numpy(rng.standard_normal((T, 2 * N, 2 * N)).astype(np.float32)).cuda()
            low = out((T, N, N))
            P.tno_mf_downsample(mf.ctx, src, 2, low)
            beta = torch.from_numpy(rng.standard_normal((6, N, N)).astype(np.float32)).cuda()
            S = torch.from_numpy(rng.standard_normal((T, n, n)).astype(np.float32)).cuda()
            gb, gs = out((6, N, N)), out((T, n, n))
            loss = P.tno_mf_scatter_lossgrad(mf.ctx, low, jit, 1.0, beta, S, gb, gs)
            torch.cuda.synchronize()
            res["low%d" % N], res["gb%d" % N], res["gs%d" % N] = (t.cpu().numpy().view(np.uint32).copy() for t in (low, gb, gs))
            res["loss%d" % N] = np.array([loss])
    return res


@pytest.mark.parametrize("T,H,W,force_generic", [(9, 64, 64, False), (12, 100, 132, False), (10, 33, 47, True)])
def test_outputs_do_not_depend_on_what_was_in_them(T, H, W, force_generic):
    """Output buffers are write-only for the library: the same calls with outputs that start as zeros and as 0xff bytes
    (NaN / -1) return the same bits -- nothing is accumulated into, or read from, an output before it is written."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    a = _all_outputs(torch, P, MatchedFilter, 0x00, T, H, W, force_generic)
    b = _all_outputs(torch, P, MatchedFilter, 0xFF, T, H, W, force_generic)
    for name in a:
        assert np.array_equal(a[name], b[name]), name
        if a[name].dtype == np.uint32 and name not in ("top", "mtop", "xtop", "t2", "t3", "ak", "a2"):
            assert np.all(np.isfinite(a[name].view(np.float32)) | np.isinf(a[name].view(np.float32))), name   # no NaN
