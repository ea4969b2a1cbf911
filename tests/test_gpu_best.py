"""GPU parity of tno_mf_best (section 3.3: max over the filter bank, scores in units of the
local standard deviation) against the CPU oracle, through the C ABI."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _run(snr, box, topk, thr):
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    d = torch.from_numpy(np.ascontiguousarray(snr, dtype=np.float32)).cuda()
    with MatchedFilter(0, topk, thr) as mf:
        mx, ak, z, top = mf.best(d, box)
        torch.cuda.synchronize()
        launches, _ = mf.stats()
        c = mf.candidates_to_numpy(top[None])[0] if top is not None else None
        return mx.cpu().numpy(), ak.cpu().numpy(), z.cpu().numpy(), c, launches


def _check(snr, box, topk=8, thr=2.0):
    mx, ak, z, c, launches = _run(snr, box, topk, thr)
    om, oa = oracle.best(snr)
    assert np.array_equal(mx, om) and np.array_equal(ak, oa)              # exact: comparisons only
    oz, _ = oracle.local_z(om, box)
    assert np.all(np.abs(z.astype(np.float64) - oz) <= 2e-6 * np.maximum(1.0, np.abs(oz)))
    assert launches >= 4
    # the list is exactly the sort of the GPU's own Z map, and carries the arg-max trajectory
    ref = oracle.topk(z.astype(np.float64), topk, thr, 0)
    assert np.array_equal(c["x"], ref["x"]) and np.array_equal(c["y"], ref["y"])
    assert np.array_equal(c["snr"].astype(np.float64), ref["snr"])
    n = int(np.count_nonzero(c["x"] >= 0))
    assert np.array_equal(c["k"][:n], ak[c["y"][:n], c["x"][:n]]) and np.all(c["k"][n:] == -1)
    return z


@pytest.mark.parametrize("shape,box", [((5, 64, 64), 9), ((3, 70, 132), 255), ((1, 33, 47), 5),
                                       ((12, 300, 260), 255), ((2, 1, 1), 3), ((4, 513, 17), 31)])
def test_best_matches_oracle(shape, box):
    rng = np.random.default_rng(sum(shape) + box)
    snr = rng.standard_normal(shape).astype(np.float32)
    snr[0, shape[1] // 2, shape[2] // 2] += 9.0
    _check(snr, box)


def test_ties_constant_maps_and_offsets():
    rng = np.random.default_rng(1)
    snr = rng.integers(-2, 3, size=(6, 40, 48)).astype(np.float32)       # exact ties: smallest k wins
    _check(snr, 7)
    const = np.full((3, 32, 32), 1.5, np.float32)                        # zero variance -> Z = 0
    z = _check(const, 5)
    assert np.all(z == 0)
    off = (rng.standard_normal((4, 96, 96)) + 1000.0).astype(np.float32)  # large mean, small spread
    _check(off, 31, thr=1e9)


def test_best_on_a_search_result_and_errors():
    """End to end: search config 2, then the paper's scoring on the maps."""
    torch = _torch()
    import tno_synth
    from helpers import cpu_inputs
    from paper_2209_09848_b200 import MatchedFilter, TnoMfError, tno_mf_best
    cfg = tno_synth.CONFIGS[2]
    p, f = cpu_inputs(cfg)
    with MatchedFilter(0, 10, 3.0) as mf:
        maps, _ = mf.search(torch.from_numpy(f).cuda(), p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0)
        mx, ak, z, top = mf.best(maps, 255)
        torch.cuda.synchronize()
        g = maps.cpu().numpy()
        om, oa = oracle.best(g)
        assert np.array_equal(mx.cpu().numpy(), om) and np.array_equal(ak.cpu().numpy(), oa)
        oz, _ = oracle.local_z(om, 255)
        assert np.abs(z.cpu().numpy() - oz).max() <= 2e-6 * max(1.0, np.abs(oz).max())
        c = mf.candidates_to_numpy(top[None])[0]
        ref = oracle.topk(z.cpu().numpy().astype(np.float64), 10, 3.0, 0)
        assert np.array_equal(c["x"], ref["x"]) and np.array_equal(c["y"], ref["y"])
        with pytest.raises(TnoMfError):
            tno_mf_best(mf.ctx, maps, 254, mx)                               # even box


def test_flux_estimate_matches_oracle_n_over_d():
    """tno_mf_flux: A = N / D, from the maps and D tables of the preceding search."""
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter, TnoMfError, tno_mf_flux
    T, H, W = 50, 96, 128
    rng = np.random.default_rng(21)
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.array([[0.2, -0.1, 0, 0], [0.2, 0.3, 0, 0.002], [-0.6, 0.0, 0, 0], [0.0, 0.0, 0, 0]], np.float32)
    amp = 2.25
    oracle.inject(f, traj[1:2], [70], [40], [amp], 1.0, 25.0)
    _, oN, oD = oracle.snr_map(f, sigma, traj, 1.0, 25.0, return_ND=True)
    ref = np.where(oD > 0, oN / np.where(oD > 0, oD, 1.0), 0.0)
    with MatchedFilter(0, 0) as mf:
        with pytest.raises(TnoMfError):                                   # no search yet on this context
            tno_mf_flux(mf.ctx, torch.zeros((4, H, W), device="cuda"), torch.zeros((4, H, W), device="cuda"))
        maps, _ = mf.search(torch.from_numpy(f).cuda(), sigma, traj, 1.0, 25.0)
        fl = mf.flux(maps)
        torch.cuda.synchronize()
        g = fl.cpu().numpy().astype(np.float64)
        with pytest.raises(TnoMfError):                                   # shape of another search
            tno_mf_flux(mf.ctx, maps[:2].contiguous(), fl[:2].contiguous())
    # |dSNR| <= 1e-3 scaled by D^(-1/2), plus float32 rounding of the product
    tol = 1e-3 / np.sqrt(np.where(oD > 0, oD, 1.0)) + 4e-7 * np.abs(ref)
    assert np.all(np.abs(g - ref) <= tol)
    # the injected amplitude is recovered at the source (noise: sigma_A = D^(-1/2))
    assert abs(g[1, 40, 70] - amp) <= 5.0 / np.sqrt(oD[1, 40, 70])
    # corner pixels, where D is clipped: still N / D
    assert g[2, 0, 0] == pytest.approx(ref[2, 0, 0], abs=float(tol[2, 0, 0]))
