"""tno_mf_local_z_static -- the entry point that allocates no device memory (scratch in a static device array of the
library, include/tno_mf.h) -- against the existing path, tno_mf_best's out_z, on consecutive calls through the C ABI.
Collected last on purpose (the file name sorts after every other test file): the suite runs with pytest -x."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

BOX = 31
MAX_PX = 1 << 20                       # the limit stated in include/tno_mf.h


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _score(shape, seed):
    """A max map: half-normal noise with a few bright peaks (what tno_mf_best / tno_mf_search_max put out)."""
    rng = np.random.default_rng(seed)
    m = np.abs(rng.standard_normal(shape)).astype(np.float32) + 2.0
    for _ in range(5):
        m[rng.integers(0, shape[0]), rng.integers(0, shape[1])] += 8.0
    return m


def _existing(P, torch, ctx, d_score, box):
    """Z through the existing path: tno_mf_best on the map as a bank of one trajectory (scratch from cudaMalloc)."""
    mx = torch.empty_like(d_score)
    z = torch.empty_like(d_score)
    P.tno_mf_best(ctx, d_score[None], box, mx, None, z, None)
    return mx, z


def test_static_scratch_matches_the_existing_path_on_consecutive_calls():
    torch = _torch()
    import paper_2209_09848_b200 as P
    ctx = P.tno_mf_create(0, None, 0, 0.0)
    try:
        # big, then small (the scratch still holds the big map's tables beyond the small one's), then ragged, then big
        shapes = [(300, 260), (70, 132), (33, 47), (513, 17), (1024, 1024), (300, 260)]
        maps = [torch.from_numpy(_score(s, 11 + i)).cuda() for i, s in enumerate(shapes)]
        ref = []
        for d in maps:
            mx, z = _existing(P, torch, ctx, d, BOX)
            torch.cuda.synchronize()
            assert torch.equal(mx, d)
            ref.append(z)
        outs = [torch.full_like(d, float("nan")) for d in maps]
        # first call on this device: resolves the address of the static array (and makes the driver load its module)
        P.tno_mf_local_z_static(ctx, maps[0], BOX, outs[0])
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        for d, o in zip(maps, outs):                       # calls in a row on one stream, no sync in between
            P.tno_mf_local_z_static(ctx, d, BOX, o)
            assert P.tno_mf_last_stats(ctx)[0] == 3
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0, "device memory changed across calls that must not allocate"
        for s, o, r in zip(shapes, outs, ref):
            a, b = o.cpu().numpy().astype(np.float64), r.cpu().numpy().astype(np.float64)
            assert np.all(np.isfinite(a))
            # the tolerance the Z tests use (tests/test_gpu_best.py) ...
            assert np.all(np.abs(a - b) <= 2e-6 * np.maximum(1.0, np.abs(b))), s
            # ... and in fact the same bits: the same arithmetic in the same order
            assert np.array_equal(o.cpu().numpy(), r.cpu().numpy()), s
        # and both against the oracle on the small maps
        for i in (1, 2, 3):
            oz, _ = oracle.local_z(maps[i].cpu().numpy(), BOX)
            a = outs[i].cpu().numpy().astype(np.float64)
            assert np.all(np.abs(a - oz) <= 2e-6 * np.maximum(1.0, np.abs(oz)))
    finally:
        P.tno_mf_destroy(ctx)


def test_static_scratch_limit_and_argument_errors():
    torch = _torch()
    import paper_2209_09848_b200 as P
    ctx = P.tno_mf_create(0, None, 0, 0.0)
    try:
        big = torch.zeros((1024, 1025), dtype=torch.float32, device="cuda")          # one column beyond the limit
        assert big.numel() > MAX_PX
        with pytest.raises(P.TnoMfError) as e:
            P.tno_mf_local_z_static(ctx, big, BOX, torch.empty_like(big))
        assert e.value.code == -1 and "1048576" in str(e.value) and "tno_mf_best" in str(e.value)
        ok = torch.ones((1, MAX_PX), dtype=torch.float32, device="cuda")             # exactly the limit, one row
        out = torch.empty_like(ok)
        P.tno_mf_local_z_static(ctx, ok, 3, out)
        torch.cuda.synchronize()
        assert torch.all(out == 0)                                                   # constant map: zero variance
        small = torch.ones((8, 8), dtype=torch.float32, device="cuda")
        with pytest.raises(P.TnoMfError) as e:
            P.tno_mf_local_z_static(ctx, small, 4, torch.empty_like(small))          # even box
        assert e.value.code == -1
        with pytest.raises(P.TnoMfError) as e:
            P.tno_mf_local_z_static(ctx, small, 3, small)                            # aliased output
        assert e.value.code == -1
    finally:
        P.tno_mf_destroy(ctx)
