"""The context's stream (include/tno_mf.h: "enqueue their work on the context's stream"): the same calls on a
non-blocking user stream, fed by work that is still running on that stream when the call is made, return the bits of
the default-stream run.  A library operation issued on any other stream would run ahead of its inputs here."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _run(torch, P, MatchedFilter, T=24, H=96, W=128):
    rng = np.random.default_rng(5)
    base = torch.from_numpy(rng.standard_normal((T, H, W)).astype(np.float32)).cuda(non_blocking=True)
    jit = (0.2 * rng.standard_normal((T, 2))).astype(np.float32)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    trajs = np.array([[0.1, -0.2, 0, 0], [0.1, 0.2, 0, 0], [0.1, 0.15, 0, 0.001], [-0.3, 0.05, 0, 0]], np.float32)
    res = {}
    with MatchedFilter(0, 6, 2.0) as mf:
        # the inputs are produced on the current stream right before each call, without a synchronisation
        big = torch.randn((64, 1024, 1024), device="cuda", generator=torch.Generator(device="cuda").manual_seed(1))
        frames = base + 0.0 * big.sum()                         # a long reduction first, then the frames
        valid = (torch.ones_like(frames) - (frames > 2.5).float()) + 0.0 * big.mean()
        mf.inject(frames, trajs[:2], np.array([40, 70]), np.array([30, 60]), np.array([6.0, 5.0]), 1.0, T / 2.0)
        maps, top = mf.search(frames, sigma, trajs, 1.0, T / 2.0)
        mmaps, mtop = mf.search(frames, sigma, trajs, 1.0, T / 2.0, valid=valid, jitter_xy=jit)
        mx, ak, _, xtop = mf.search_max(frames, sigma, trajs, 1.0, T / 2.0)
        flux = mf.flux(maps)
        m2, a2, z, t2 = mf.best(maps, 9)
        zs = torch.empty_like(z)
        P.tno_mf_local_z_static(mf.ctx, m2, 9, zs)
        pk, t3 = mf.peaks(z, 3, a2)
        coef, resid = mf.background(frames * 1.0, jit, 1.0, 3)
        low = torch.empty((T, H // 2, W // 2), device="cuda")
        P.tno_mf_downsample(mf.ctx, frames, 2, low)
        sq = (frames[:, :64, :64] * 1.0).contiguous()
        beta = torch.zeros((6, 64, 64), device="cuda") + 0.1
        S = torch.zeros((T, 8, 8), device="cuda") + 0.2
        gb, gs = torch.empty_like(beta), torch.empty_like(S)
        loss = P.tno_mf_scatter_lossgrad(mf.ctx, sq, jit, 1.0, beta, S, gb, gs)
        fl, it, ev = P.tno_mf_scatter_fit(mf.ctx, sq, jit, 1.0, 10, 0.0, beta, S)
        # host entry point: its copy streams must wait for nothing but their own uploads
        host = base.cpu().numpy()
        hmaps = np.empty((4, H, W), np.float32)
        mf.search_host(host, sigma, trajs, 1.0, T / 2.0, out_snr_host=hmaps)
        torch.cuda.current_stream().synchronize()
        for name, t in (("maps", maps), ("top", top), ("mmaps", mmaps), ("mtop", mtop), ("mx", mx), ("ak", ak), ("xtop", xtop),
                        ("flux", flux), ("m2", m2), ("a2", a2), ("z", z), ("t2", t2), ("zs", zs), ("pk", pk), ("t3", t3),
                        ("coef", coef), ("resid", resid), ("low", low), ("gb", gb), ("gs", gs), ("beta", beta), ("S", S)):
            res[name] = t.cpu().numpy()
        res["hmaps"] = hmaps
        res["scalars"] = np.array([loss, fl, it, ev])
    return res


def test_calls_on_a_user_stream_match_the_default_stream():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2209_09848_b200 as P
    from paper_2209_09848_b200 import MatchedFilter
    ref = _run(torch, P, MatchedFilter)
    s = torch.cuda.Stream()                       # non-blocking: does not synchronise with the legacy default stream
    with torch.cuda.stream(s):
        out = _run(torch, P, MatchedFilter)
    s.synchronize()
    for name in ref:
        assert np.array_equal(ref[name], out[name], equal_nan=True), name
    assert np.all(np.isfinite(out["maps"])) and np.all(np.isfinite(out["gs"]))


def test_two_contexts_on_two_streams_are_independent():
    """include/tno_mf.h: "distinct contexts are independent".  Two contexts on two non-blocking streams, different banks
    and stacks, their calls issued alternately without any synchronisation, against each run alone."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2209_09848_b200 import MatchedFilter
    rng = np.random.default_rng(9)
    T, H, W = 40, 192, 256
    fa = torch.from_numpy(rng.standard_normal((T, H, W)).astype(np.float32)).cuda()
    fb = torch.from_numpy(rng.standard_normal((T, H, W)).astype(np.float32)).cuda()
    sigma = np.ones(T, np.float32)
    ta = np.array([[0.1, -0.2, 0, 0], [0.1, 0.2, 0, 0], [-0.3, 0.05, 0, 0]], np.float32)
    tb = np.array([[0.25, 0.3, 0, 0], [0.25, -0.3, 0, 0], [0.25, 0.1, 0, 0.002], [0.0, 0.0, 0, 0]], np.float32)

    def alone(f, tr):
        with MatchedFilter(0, 5, 2.0) as mf:
            maps, top = mf.search(f, sigma, tr, 1.0, T / 2.0)
            mx, ak, z, _ = mf.best(maps, 9)
            torch.cuda.synchronize()
            return [t.cpu().numpy() for t in (maps, top, mx, ak, z)]

    ra, rb = alone(fa, ta), alone(fb, tb)
    torch.cuda.synchronize()
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    with torch.cuda.stream(sa):
        ma = MatchedFilter(0, 5, 2.0)
    with torch.cuda.stream(sb):
        mb = MatchedFilter(0, 5, 2.0)
    outs_a, outs_b = [], []
    for rep in range(3):                                   # alternately, nothing waits for anything
        with torch.cuda.stream(sa):
            maps, top = ma.search(fa, sigma, ta, 1.0, T / 2.0)
            outs_a.append((maps, top) + ma.best(maps, 9)[:3])
        with torch.cuda.stream(sb):
            maps, top = mb.search(fb, sigma, tb, 1.0, T / 2.0)
            outs_b.append((maps, top) + mb.best(maps, 9)[:3])
    sa.synchronize()
    sb.synchronize()
    for outs, ref in ((outs_a, ra), (outs_b, rb)):
        for o in outs:
            for t, r in zip(o, ref):
                assert np.array_equal(t.cpu().numpy(), r)
    ma.close()
    mb.close()
