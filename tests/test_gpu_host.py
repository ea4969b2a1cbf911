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
