"""Shared helpers of the GPU parity tests: build a config's inputs, run the CUDA library, and
compare with the CPU oracle under the acceptance rules of DESIGN.md (readings c15, c16)."""
import numpy as np

import oracle
import tno_synth

TOL = 1e-3          # BASELINE.json:north_star "|dSNR| <= 1e-3 absolute"


def cpu_inputs(cfg):
    """(params, float32 stack with sources injected by the ORACLE's renderer)."""
    p = tno_synth.make_params(cfg)
    f = tno_synth.stack_numpy(p)
    if len(p.src_k):
        oracle.inject(f, p.traj[p.src_k], p.src_x, p.src_y, p.src_amp, cfg.prf_sigma, cfg.t0)
    return p, f


def run_gpu(frames_dev, sigma_t, traj, prf_sigma, t0, topk, threshold, want_maps=True,
            force_generic=False, sep_shape=0):
    """-> (maps float32 [K,H,W] numpy or None, candidates structured [K,topk] or None, stats)."""
    import torch
    from paper_2209_09848_b200 import MatchedFilter
    with MatchedFilter(frames_dev.device.index or 0, topk, threshold, force_generic, sep_shape=sep_shape) as mf:
        maps, cand = mf.search(frames_dev, sigma_t, traj, prf_sigma, t0, want_maps=want_maps)
        torch.cuda.synchronize()
        stats = mf.stats()
        m = maps.cpu().numpy() if maps is not None else None
        c = mf.candidates_to_numpy(cand) if cand is not None else None
    return m, c, stats


def check_topk(gpu, omap, k, ktop, thr, tol=TOL):
    """Acceptance of one trajectory's GPU list against the oracle map (DESIGN.md c15)."""
    assert gpu.shape == (ktop,)
    assert np.all(gpu["k"] == k)
    nvalid = int(np.count_nonzero(gpu["x"] >= 0))
    v, pad = gpu[:nvalid], gpu[nvalid:]
    assert np.all(v["x"] >= 0) and np.all(v["y"] >= 0)
    assert np.all(pad["x"] == -1) and np.all(pad["y"] == -1) and np.all(np.isneginf(pad["snr"]))
    pix = v["y"].astype(np.int64) * omap.shape[1] + v["x"]
    assert len(np.unique(pix)) == nvalid, "duplicate candidates"
    o_at = omap[v["y"], v["x"]]
    assert np.all(np.abs(v["snr"].astype(np.float64) - o_at) <= tol)           # (i)
    above = np.sort(omap[omap >= thr])[::-1]
    tau = max(above[ktop - 1] if above.size >= ktop else thr, thr)
    assert np.all(o_at >= tau - tol)                                            # (ii)
    must_y, must_x = np.nonzero(omap > tau + tol)                                # (iii)
    got = set(pix.tolist())
    for yy, xx in zip(must_y, must_x):
        assert int(yy) * omap.shape[1] + int(xx) in got, ("missing", k, xx, yy, omap[yy, xx])
    s = v["snr"]
    assert np.all(s[:-1] >= s[1:])                                               # (iv)
    eq = np.nonzero(s[:-1] == s[1:])[0]
    assert np.all(pix[eq] < pix[eq + 1]), "exact ties must be ordered by (y, x)"
    n_sure = int(np.count_nonzero(omap > thr + tol))
    n_maybe = int(np.count_nonzero(omap >= thr - tol))
    assert min(n_sure, ktop) <= nvalid <= min(n_maybe, ktop)


def check_topk_vs_own_map(gpu, gmap, k, ktop, thr):
    """The GPU list must equal, exactly, the plain sort of the GPU's own float32 map."""
    ref = oracle.topk(gmap.astype(np.float64), ktop, thr, k)
    assert np.array_equal(gpu["x"], ref["x"]) and np.array_equal(gpu["y"], ref["y"])
    assert np.array_equal(gpu["snr"].astype(np.float64), ref["snr"])
    assert np.all(gpu["k"] == k)


def scatter_problem(seed, T, N, n, noise=0.3, outliers=0.02):
    """Smooth scattered light that changes from frame to frame over a static background that moves with the
    jitter, plus noise and a few outliers (the shape of the paper's problem)."""
    rng = np.random.default_rng(seed)
    jit = (0.15 * rng.standard_normal((T, 2))).astype(np.float32)
    beta = rng.standard_normal((6, N, N)) * np.array([20, 3, 3, 1, 1, 1])[:, None, None]
    S = 10.0 + 5.0 * rng.standard_normal((T, n, n))
    D = oracle.upsample(S, N) + np.einsum("tk,kij->tij", oracle.background_basis(jit), beta)
    D += noise * rng.standard_normal(D.shape)
    D += (rng.uniform(size=D.shape) < outliers) * rng.laplace(0, 15, size=D.shape)
    return D.astype(np.float32), jit, beta, S


