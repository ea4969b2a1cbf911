"""tno_mf_search_host: stack in host memory, banded upload overlapped with the search, results to host
memory -- bit for bit the results of the device-pointer call."""
import numpy as np
import pytest

from helpers import run_gpu

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.mark.parametrize("shape,pinned", [((12, 1024, 256), True), ((12, 1024, 256), False), ((30, 200, 64), True),
                                          ((5, 33, 47), True), ((3, 2500, 128), True)])
def test_host_search_equals_device_search(shape, pinned):
    torch = _torch()
    import paper_2209_09848_b200 as P
    T, H, W = shape
    rng = np.random.default_rng(T + H + W)
    f = torch.from_numpy(rng.standard_normal(shape).astype(np.float32))
    if pinned:
        f = f.pin_memory()
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.array([[0.3, -0.2, 0, 0], [0.3, 0.45, 0, 0], [0.3, 0.0, 0, 0.01], [-1.25, 0.5, 0, 0],
                     [0.0, 0.0, 0, 0], [0.3, 7.0, 0, 0], [0.3, -5.5, 0, 0.2]], np.float32)   # large y-shifts too:
    n, topk = traj.shape[0], 6                   # the early finish of output rows must wait for them
    ref_m, ref_c, _ = run_gpu(f.cuda(), sigma, traj, 1.0, T / 2.0, topk, 3.0)
    ctx = P.tno_mf_create(0, None, topk, 3.0)
    out = torch.empty((n, H, W), dtype=torch.float32)
    cand = np.zeros((n, topk), dtype=P.CAND_DTYPE)
    if pinned:
        out = out.pin_memory()
    for _ in range(2):                                     # the second call reuses the context's device stack
        out.zero_()
        P.tno_mf_search_host(ctx, f, sigma, None, None, traj, 1.0, T / 2.0, out, cand)
        assert np.array_equal(out.numpy(), ref_m)
        assert np.array_equal(cand, ref_c)
    # lists only, and with frame times / jitter through the same path
    cand2 = np.zeros((n, topk), dtype=P.CAND_DTYPE)
    P.tno_mf_search_host(ctx, f, sigma, None, None, traj, 1.0, T / 2.0, None, cand2)
    assert np.array_equal(cand2, ref_c)
    times = np.cumsum(rng.uniform(0.5, 1.5, T)).astype(np.float32)
    jit = rng.uniform(-1, 1, (T, 2)).astype(np.float32)
    P.tno_mf_search_host(ctx, f, sigma, times, jit, traj, 1.0, float(times[T // 2]), out, None)
    d_out = torch.empty((n, H, W), device="cuda")
    P.tno_mf_search_ex(ctx, f.cuda(), sigma, times, jit, traj, 1.0, float(times[T // 2]), d_out)
    torch.cuda.synchronize()
    assert np.array_equal(out.numpy(), d_out.cpu().numpy())
    with pytest.raises(P.TnoMfError):
        P.tno_mf_search_host(ctx, f, sigma, None, None, traj, 1.0, 0.0, None, None)
    P.tno_mf_destroy(ctx)


def test_early_finish_with_all_negative_y_shifts():
    """Every y-shift negative (t0 before the first frame, all vy < 0): the banded early finish reaches the last
    output row before the last band; the final finish launch must then be skipped, not launched empty."""
    torch = _torch()
    import paper_2209_09848_b200 as P
    T, H, W = 8, 640, 128
    rng = np.random.default_rng(12)
    f = torch.from_numpy(rng.standard_normal((T, H, W)).astype(np.float32)).pin_memory()
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.array([[0.2, -4.0, 0, 0], [0.2, -6.5, 0, 0], [-0.1, -5.0, 0, -0.1]], np.float32)
    t0 = -10.0                                             # dt = 10 .. 17: shifts -40 .. -140
    n, topk = traj.shape[0], 5
    ctx = P.tno_mf_create(0, None, topk, 3.0)
    d_out = torch.empty((n, H, W), device="cuda")
    d_top = torch.empty((n, topk, 4), dtype=torch.int32, device="cuda")
    P.tno_mf_search_ex(ctx, f.cuda(), sigma, None, None, traj, 1.0, t0, d_out, d_top)
    torch.cuda.synchronize()
    assert P.tno_mf_last_stats(ctx)[1] == 1
    out = torch.empty((n, H, W), dtype=torch.float32).pin_memory()
    cand = np.zeros((n, topk), dtype=P.CAND_DTYPE)
    P.tno_mf_search_host(ctx, f, sigma, None, None, traj, 1.0, t0, out, cand)
    assert P.tno_mf_last_stats(ctx)[1] == 1
    assert np.array_equal(out.numpy(), d_out.cpu().numpy())
    assert np.array_equal(cand.view(np.int32).reshape(n, topk, 4), d_top.cpu().numpy())
    P.tno_mf_destroy(ctx)


@pytest.mark.parametrize("shape,masked", [((10, 700, 192), False), ((10, 700, 192), True), ((6, 40, 36), True),
                                          ((4, 50, 30), True)])
def test_host_search_with_mask_and_fused_max(shape, masked):
    """tno_mf_search_host_max: validity weights and the max over the bank through the host entry point, bit for bit
    the results of tno_mf_search_max on the uploaded stacks (banded finish with two passes; generic path for W=30)."""
    torch = _torch()
    import paper_2209_09848_b200 as P
    T, H, W = shape
    rng = np.random.default_rng(H + W)
    valid = (rng.uniform(size=shape) > 0.05).astype(np.float32)
    fr = rng.standard_normal(shape).astype(np.float32) * valid
    f, v = torch.from_numpy(fr).pin_memory(), torch.from_numpy(valid).pin_memory()
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.array([[0.3, -0.2, 0, 0], [0.3, 0.45, 0, 0], [0.3, 2.5, 0, 0], [-1.25, 0.5, 0, 0], [0.0, 0.0, 0, 0],
                     [0.3, -3.5, 0, 0.1]], np.float32)
    n, topk = traj.shape[0], 7
    ctx = P.tno_mf_create(0, None, topk, 2.5)
    dv = v.cuda() if masked else None
    d_max = torch.empty((H, W), device="cuda")
    d_arg = torch.empty((H, W), dtype=torch.int32, device="cuda")
    d_out = torch.empty((n, H, W), device="cuda")
    d_top = torch.empty((n, topk, 4), dtype=torch.int32, device="cuda")
    P.tno_mf_search_max(ctx, f.cuda(), dv, sigma, None, None, traj, 1.0, T / 2.0, d_max, d_arg, d_out, d_top)
    torch.cuda.synchronize()
    h_max = torch.empty((H, W)).pin_memory()
    h_arg = torch.empty((H, W), dtype=torch.int32).pin_memory()
    h_out = torch.empty((n, H, W)).pin_memory()
    cand = np.zeros((n, topk), dtype=P.CAND_DTYPE)
    for _ in range(2):
        h_out.zero_(); h_max.zero_()
        P.tno_mf_search_host_max(ctx, f, v if masked else None, sigma, None, None, traj, 1.0, T / 2.0, h_max, h_arg,
                                 h_out, cand)
        assert torch.equal(h_max, d_max.cpu()) and torch.equal(h_arg, d_arg.cpu())
        assert torch.equal(h_out, d_out.cpu())
        assert np.array_equal(cand.view(np.int32).reshape(n, topk, 4), d_top.cpu().numpy())
    # the max map as the only output
    h_max.zero_()
    P.tno_mf_search_host_max(ctx, f, v if masked else None, sigma, None, None, traj, 1.0, T / 2.0, h_max, None, None, None)
    assert torch.equal(h_max, d_max.cpu())
    with pytest.raises(P.TnoMfError):
        P.tno_mf_search_host_max(ctx, f, None, sigma, None, None, traj, 1.0, 0.0, None, h_arg, None, None)
    with pytest.raises(AssertionError):                       # undersized host buffer is caught by the binding
        P.tno_mf_search_host_max(ctx, f, None, sigma, None, None, traj, 1.0, 0.0, h_max, None, h_out[:2], None)
    P.tno_mf_destroy(ctx)


def test_host_search_at_full_size_equals_device_search():
    """The launch bench.py's e2e leg times (config 3: 9 bands of 4 tile rows, early finish, banded download):
    maps and lists bit for bit those of the device search."""
    torch = _torch()
    import tno_synth
    from paper_2209_09848_b200 import MatchedFilter
    cfg = tno_synth.CONFIGS[3]
    p = tno_synth.make_params(cfg)
    dev = torch.device("cuda", 0)
    frames = tno_synth.stack_torch(p, dev)
    mf = MatchedFilter(0, cfg.topk, cfg.threshold)
    mf.inject(frames, p.traj[p.src_k], p.src_x, p.src_y, p.src_amp, cfg.prf_sigma, cfg.t0)
    maps, cand = mf.search(frames, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0)
    torch.cuda.synchronize()
    host = torch.empty(frames.shape, dtype=torch.float32, pin_memory=True)
    host.copy_(frames)
    del frames
    h_snr = torch.empty(maps.shape, dtype=torch.float32, pin_memory=True)
    h_top = torch.empty(cand.shape, dtype=torch.int32, pin_memory=True)
    mf.search_host(host, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0, h_snr, h_top)
    assert mf.stats()[1] == 1
    assert torch.equal(h_top, cand.cpu())
    for k0 in range(0, cfg.n_traj, 10):
        assert torch.equal(h_snr[k0:k0 + 10], maps[k0:k0 + 10].cpu())
    mf.close()
