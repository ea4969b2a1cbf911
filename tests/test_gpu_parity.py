"""GPU parity: the CUDA library (through its C ABI) against the CPU oracle, element by element.
Run on a B200 with `pytest -m gpu`."""
import numpy as np
import pytest

import oracle
import tno_synth
from helpers import TOL, check_topk, check_topk_vs_own_map, cpu_inputs, run_gpu

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


def _compare_full(cfg, force_generic):
    torch = _torch()
    p, f = cpu_inputs(cfg)
    om = oracle.snr_map(f, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0)
    fd = torch.from_numpy(f).cuda()
    gm, gc, stats = run_gpu(fd, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0, cfg.topk, cfg.threshold,
                            force_generic=force_generic)
    assert stats[1] == (0 if force_generic else 1)
    assert stats[0] >= 5
    err = np.abs(gm.astype(np.float64) - om)
    assert err.max() <= TOL, (err.max(), np.unravel_index(err.argmax(), err.shape))
    for k in range(cfg.n_traj):
        check_topk(gc[k], om[k], k, cfg.topk, cfg.threshold)
        check_topk_vs_own_map(gc[k], gm[k], k, cfg.topk, cfg.threshold)
    # injected sources are where the oracle says they are
    for i in range(len(p.src_k)):
        k, x, y = int(p.src_k[i]), int(p.src_x[i]), int(p.src_y[i])
        assert abs(float(gm[k, y, x]) - om[k, y, x]) <= TOL
    return err.max()


@pytest.mark.parametrize("force_generic", [False, True])
def test_config1_full_maps_and_topk(force_generic):
    _compare_full(tno_synth.CONFIGS[1], force_generic)


@pytest.mark.parametrize("force_generic", [False, True])
def test_config2_full_maps_and_topk(force_generic):
    _compare_full(tno_synth.CONFIGS[2], force_generic)


def test_config1_against_oracle_point_everywhere():
    torch = _torch()
    cfg = tno_synth.CONFIGS[1]
    p, f = cpu_inputs(cfg)
    gm, _, _ = run_gpu(torch.from_numpy(f).cuda(), p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0,
                       cfg.topk, cfg.threshold)
    for k in range(cfg.n_traj):
        for y in range(0, cfg.H, 3):
            for x in range(0, cfg.W, 3):
                s, _, _ = oracle.point(f, p.sigma_t, p.traj[k], cfg.prf_sigma, cfg.t0, x, y)
                assert abs(float(gm[k, y, x]) - s) <= TOL


@pytest.mark.parametrize("shape,force_generic", [
    ((7, 64, 64), False), ((3, 70, 132), False), ((5, 130, 68), False), ((1, 8, 8), False),
    ((4, 33, 47), True), ((2, 1, 1), True), ((3, 5, 9), True), ((6, 65, 4), False),
    ((70, 40, 72), False),
])
def test_ragged_shapes_and_mixed_trajectories(shape, force_generic):
    """Sizes that are not multiples of the tile, tiny frames, T < pipeline depth, T > one flush
    segment; trajectories with shared and unshared x-motions, accelerations, exact ties."""
    torch = _torch()
    T, H, W = shape
    rng = np.random.default_rng(T * 10007 + H * 101 + W)
    f = rng.standard_normal(shape).astype(np.float32)
    f[T // 2, H // 2, W // 2] += 40.0
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.array([[0.3, -0.2, 0, 0], [0.3, 0.45, 0, 0], [0.3, 0.0, 0, 0.01], [-1.25, 0.5, 0, 0],
                     [0.5, 0.5, 0, 0], [-0.5, 0.25, 0, 0], [0, 0, 0, 0], [2.0, -3.0, 0.1, 0],
                     [0.3, -0.2, 0, 0], [0.11, 0.9, -0.02, 0.03], [0.3, 7.0, 0, 0]], dtype=np.float32)
    t0 = float(T // 2)
    om = oracle.snr_map(f, sigma, traj, 1.0, t0)
    gm, gc, stats = run_gpu(torch.from_numpy(f).cuda(), sigma, traj, 1.0, t0, 7, 2.5,
                            force_generic=force_generic)
    if W % 4 != 0:
        assert stats[1] == 0        # shapes the TMA kernel does not take go to the generic kernel
    err = np.abs(gm.astype(np.float64) - om)
    assert err.max() <= TOL, (err.max(), np.unravel_index(err.argmax(), err.shape))
    for k in range(traj.shape[0]):
        check_topk(gc[k], om[k], k, 7, 2.5)
        check_topk_vs_own_map(gc[k], gm[k], k, 7, 2.5)


@pytest.mark.parametrize("offset_floats", [1, 2, 3])
def test_frames_pointer_not_16_byte_aligned_takes_the_generic_kernel(offset_floats):
    """SURVEY 8(b) shape rule: the TMA path needs a 16-byte aligned `frames`; a stack that starts 4, 8 or 12 bytes
    past such a boundary (a view into a larger buffer) must take the generic kernel and give the same answer.  The
    validity weights of a masked search fall under the same rule."""
    torch = _torch()
    import paper_2209_09848_b200 as P
    T, H, W = 9, 72, 64
    rng = np.random.default_rng(offset_floats)
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.array([[0.3, -0.2, 0, 0], [0.3, 0.45, 0, 0], [-1.25, 0.5, 0, 0.02], [0, 0, 0, 0]], np.float32)
    om = oracle.snr_map(f, sigma, traj, 1.0, 4.0)
    buf = torch.zeros(T * H * W + 8, dtype=torch.float32, device="cuda")
    assert buf.data_ptr() % 16 == 0
    view = buf[offset_floats:offset_floats + T * H * W].view(T, H, W)
    view.copy_(torch.from_numpy(f))
    assert view.data_ptr() % 16 == 4 * offset_floats and view.is_contiguous()
    gm, gc, stats = run_gpu(view, sigma, traj, 1.0, 4.0, 6, 2.5)
    assert stats[1] == 0, "an unaligned stack must not go to the TMA kernel"
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
    for k in range(traj.shape[0]):
        check_topk(gc[k], om[k], k, 6, 2.5)
    # aligned frames, unaligned validity weights
    ctx = P.tno_mf_create(0, None, 0, 0.0)
    fd = torch.from_numpy(f).cuda()
    vbuf = torch.ones(T * H * W + 8, dtype=torch.float32, device="cuda")
    valid = vbuf[offset_floats:offset_floats + T * H * W].view(T, H, W)
    out = torch.empty((4, H, W), device="cuda")
    P.tno_mf_search_masked(ctx, fd, valid, sigma, None, None, traj, 1.0, 4.0, out, None)
    torch.cuda.synchronize()
    assert P.tno_mf_last_stats(ctx)[1] == 0
    assert np.abs(out.cpu().numpy().astype(np.float64) - om).max() <= TOL
    P.tno_mf_destroy(ctx)


def test_zero_frames_and_threshold_edges():
    torch = _torch()
    T, H, W = 5, 64, 64
    z = torch.zeros((T, H, W), device="cuda")
    sigma = np.ones(T, np.float32)
    traj = np.array([[0.2, 0.1, 0, 0], [7.0, 0, 0, 0]], np.float32)
    gm, gc, _ = run_gpu(z, sigma, traj, 1.0, 2.0, 4, 5.0)
    assert np.all(gm == 0.0)
    assert np.all(gc["x"] == -1) and np.all(np.isneginf(gc["snr"]))
    # threshold -inf: every pixel competes; lists are full and start at pixel (0, 0) on all-zero maps
    gm, gc, _ = run_gpu(z, sigma, traj, 1.0, 2.0, 4, float("-inf"))
    assert gc["x"][0].tolist() == [0, 1, 2, 3] and gc["y"][0].tolist() == [0, 0, 0, 0]
    # maps only / lists only
    gm, gc, _ = run_gpu(z, sigma, traj, 1.0, 2.0, 0, 5.0)
    assert gc is None and gm.shape == (2, H, W)
    gm, gc, _ = run_gpu(z, sigma, traj, 1.0, 2.0, 3, 5.0, want_maps=False)
    assert gm is None and gc.shape == (2, 3)


def test_many_candidates_per_tile_and_exact_ties():
    """More candidates than K in one tile (tile-level selection), exact ties across tiles."""
    torch = _torch()
    T, H, W = 3, 128, 192
    f = np.zeros((T, H, W), np.float32)
    f[:, 10:50, 5:60] = 3.0                      # a bright plateau: hundreds of candidates, many ties
    f[:, 100, 150] = 9.0
    f[:, 100, 20] = 9.0                          # exact tie with the previous one, another tile
    sigma = np.ones(T, np.float32)
    traj = np.zeros((2, 4), np.float32)
    traj[1, 0] = 1.0
    om = oracle.snr_map(f, sigma, traj, 1.0, 1.0)
    for generic in (False, True):
        gm, gc, _ = run_gpu(torch.from_numpy(f).cuda(), sigma, traj, 1.0, 1.0, 50, 1.0,
                            force_generic=generic)
        assert np.abs(gm - om).max() <= TOL
        for k in range(2):
            check_topk_vs_own_map(gc[k], gm[k], k, 50, 1.0)
            check_topk(gc[k], om[k], k, 50, 1.0)


def test_inject_matches_oracle_renderer():
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    cfg = tno_synth.CONFIGS[2]
    p = tno_synth.make_params(cfg)
    base = tno_synth.stack_numpy(p)
    a = base.copy()
    oracle.inject(a, p.traj[p.src_k], p.src_x, p.src_y, p.src_amp, cfg.prf_sigma, cfg.t0)
    d = torch.from_numpy(base).cuda()
    with MatchedFilter(0) as mf:
        mf.inject(d, p.traj[p.src_k], p.src_x, p.src_y, p.src_amp, cfg.prf_sigma, cfg.t0)
        torch.cuda.synchronize()
    b = d.cpu().numpy()
    changed = a != base
    assert np.array_equal(b != base, changed) or np.count_nonzero((b != base) ^ changed) < 10
    # identical up to one float32 rounding of exp()
    assert np.max(np.abs(a - b)) <= 1e-6 * max(1.0, float(np.abs(a).max()))
    assert np.count_nonzero(a != b) <= 0.01 * np.count_nonzero(changed)


def test_errors_are_reported():
    torch = _torch()
    import paper_2209_09848_b200 as P
    ctx = P.tno_mf_create(0, None, 3, 5.0)
    f = torch.zeros((2, 8, 8), device="cuda")
    out = torch.empty((1, 8, 8), device="cuda")
    with pytest.raises(P.TnoMfError) as e:
        P.tno_mf_search(ctx, f, np.array([1.0, -1.0], np.float32), np.zeros((1, 4), np.float32), 1.0, 0.0, out)
    assert e.value.code == -1 and "sigma_t" in str(e.value)
    with pytest.raises(P.TnoMfError):
        P.tno_mf_search(ctx, f, np.ones(2, np.float32), np.zeros((1, 4), np.float32), 0.0, 0.0, out)
    with pytest.raises(P.TnoMfError):
        P.tno_mf_search(ctx, f, np.ones(2, np.float32), np.array([[np.nan, 0, 0, 0]], np.float32), 1.0, 0.0, out)
    with pytest.raises(P.TnoMfError):
        P.tno_mf_search(ctx, f, np.ones(2, np.float32), np.zeros((1, 4), np.float32), 1.0, 0.0, None, None)
    P.tno_mf_search(ctx, f, np.ones(2, np.float32), np.zeros((1, 4), np.float32), 1.0, 0.0, out)
    torch.cuda.synchronize()
    P.tno_mf_destroy(ctx)


def _bank_case(T, H, W, seed):
    rng = np.random.default_rng(seed)
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    f[:, H // 3, W // 3] += 6.0
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    return f, sigma


def test_chunked_workspace_gives_identical_results():
    """A workspace cap smaller than the bank's partial-sum buffer makes the library search the bank
    in chunks of whole batches; maps and lists must be bitwise those of the one-chunk search."""
    torch = _torch()
    from paper_2209_09848_b200 import MatchedFilter
    T, H, W = 40, 128, 128
    f, sigma = _bank_case(T, H, W, 11)
    vs = np.linspace(-0.3, 0.3, 6).astype(np.float32)
    traj = np.array([[vx, vy, 0, 0] for vx in vs for vy in vs], np.float32)      # 6 x-classes x 6 entries
    d = torch.from_numpy(f).cuda()
    outs = []
    for limit in (0, 1):           # 1 MiB: one batch (6 entries x 1-2 pieces x 64 KiB) per chunk
        with MatchedFilter(0, 9, 3.0, workspace_limit_mb=limit) as mf:
            maps, cand = mf.search(d, sigma, traj, 1.0, T / 2.0)
            torch.cuda.synchronize()
            launches, kernel = mf.stats()
            outs.append((maps.cpu().numpy(), mf.candidates_to_numpy(cand), launches))
        assert kernel == 1
    assert outs[1][2] > outs[0][2], "the capped search must have used more launches (chunks)"
    assert np.array_equal(outs[0][0], outs[1][0])
    assert np.array_equal(outs[0][1], outs[1][1])
    om = oracle.snr_map(f, sigma, traj, 1.0, T / 2.0)
    assert np.abs(outs[1][0] - om).max() <= TOL


def test_fast_trajectories_need_many_pieces():
    """y-shift ranges of several tile heights (many partial-sum pieces per output row), shifts that
    jump by more than one pixel per frame, accelerations that make the track come back."""
    torch = _torch()
    T, H, W = 60, 200, 64
    f, sigma = _bank_case(T, H, W, 12)
    traj = np.array([[0.0, 3.7, 0, 0], [0.0, -2.2, 0, 0], [0.0, 0.4, 0, 0.12], [0.25, 1.0, 0, -0.05],
                     [0.25, 0.0, 0, 0], [0.0, 0.0, 0, 0]], np.float32)
    om = oracle.snr_map(f, sigma, traj, 1.0, 30.0)
    gm, gc, stats = run_gpu(torch.from_numpy(f).cuda(), sigma, traj, 1.0, 30.0, 5, 3.0)
    assert stats[1] == 1
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
    for k in range(traj.shape[0]):
        check_topk(gc[k], om[k], k, 5, 3.0)
        check_topk_vs_own_map(gc[k], gm[k], k, 5, 3.0)


@pytest.mark.parametrize("sep_shape", [0, 1, 2])
def test_results_are_reproducible_and_independent_of_the_bank(sep_shape):
    """Bitwise identical maps from run to run, and the map of a trajectory does not depend on which
    other trajectories are searched with it (summation order is a function of the trajectory and of the kernel
    shape; with sep_shape = 0 the library picks the shape per call, here the same one for both banks)."""
    torch = _torch()
    T, H, W = 130, 96, 128
    f, sigma = _bank_case(T, H, W, 13)
    vs = np.linspace(-0.2, 0.2, 5).astype(np.float32)
    traj = np.array([[vx, vy, 0, 0] for vx in vs[:2] for vy in vs], np.float32)
    d = torch.from_numpy(f).cuda()
    a, _, _ = run_gpu(d, sigma, traj, 1.0, 65.0, 4, 3.0, sep_shape=sep_shape)
    b, _, _ = run_gpu(d, sigma, traj, 1.0, 65.0, 4, 3.0, sep_shape=sep_shape)
    assert np.array_equal(a, b)
    sub = np.array([0, 3, 7])
    c, _, _ = run_gpu(d, sigma, traj[sub], 1.0, 65.0, 4, 3.0, sep_shape=sep_shape)
    assert np.array_equal(a[sub], c)


@pytest.mark.parametrize("sep_shape", [1, 2])
@pytest.mark.parametrize("cfg_idx", [1, 2])
def test_both_kernel_shapes_on_configs_1_and_2(cfg_idx, sep_shape):
    """The two shapes of the separable kernel (4 positions x 5 slots, tiles of 48 rows; 5 x 4, tiles of 60 rows),
    each forced: full maps and lists against the oracle."""
    torch = _torch()
    cfg = tno_synth.CONFIGS[cfg_idx]
    p, f = cpu_inputs(cfg)
    om = oracle.snr_map(f, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0)
    gm, gc, stats = run_gpu(torch.from_numpy(f).cuda(), p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0, cfg.topk,
                            cfg.threshold, sep_shape=sep_shape)
    assert stats[1] == 1
    err = np.abs(gm.astype(np.float64) - om)
    assert err.max() <= TOL, (err.max(), np.unravel_index(err.argmax(), err.shape))
    for k in range(cfg.n_traj):
        check_topk(gc[k], om[k], k, cfg.topk, cfg.threshold)
        check_topk_vs_own_map(gc[k], gm[k], k, cfg.topk, cfg.threshold)


@pytest.mark.parametrize("sep_shape", [1, 2])
def test_mirror_pairs_edge_cases(sep_shape):
    """Slots of the separable kernel: pairs (+-vy, +-ay), a pair with exact half-pixel ties
    (must NOT share a slot: floor(-d + 1/2) != -floor(d + 1/2) there), duplicates, a lone negative motion, vy = 0 with
    and without acceleration, six slots of one x-motion (two batches).  Every map against the oracle, and every
    trajectory alone gives the same bits as inside the bank -- with or without its mirror image next to it."""
    torch = _torch()
    T, H, W = 90, 100, 128
    f, sigma = _bank_case(T, H, W, 29)
    traj = np.array([[0.3, 0.2, 0, 0], [0.3, -0.2, 0, 0],            # a pair
                     [0.3, 0.5, 0, 0], [0.3, -0.5, 0, 0],            # exact ties at odd dt: two single slots
                     [0.3, 0.2, 0, 0],                               # duplicate of the first
                     [0.3, 0.11, 0, 0.002], [0.3, -0.11, 0, -0.002],  # a pair with acceleration
                     [0.3, -0.37, 0, 0.001],                         # lone minus member (its mirror is not in the bank)
                     [0.3, 0.0, 0, 0], [0.3, 0.0, 0, 0.003], [0.3, 0.0, 0, -0.003],   # vy = 0
                     [-0.1, -0.45, 0, 0], [-0.1, 0.45, 0, 0]], np.float32)            # a second x-motion
    t0 = 45.0
    import paper_2209_09848_b200 as P
    n, batch, slot, member = P.tno_mf_plan_slots(traj, T, t0)
    assert slot[0] == slot[1] and member[0] == 0 and member[1] == 1
    assert (batch[2], slot[2]) != (batch[3], slot[3]) and member[2] == 0 and member[3] == 0      # ties: not paired
    assert member[7] == 1 and (batch[9], slot[9]) == (batch[10], slot[10])
    om = oracle.snr_map(f, sigma, traj, 1.0, t0)
    d = torch.from_numpy(f).cuda()
    gm, gc, stats = run_gpu(d, sigma, traj, 1.0, t0, 6, 3.0, sep_shape=sep_shape)
    assert stats[1] == 1
    err = np.abs(gm.astype(np.float64) - om)
    assert err.max() <= TOL, (err.max(), np.unravel_index(err.argmax(), err.shape))
    for k in range(traj.shape[0]):
        check_topk(gc[k], om[k], k, 6, 3.0)
        check_topk_vs_own_map(gc[k], gm[k], k, 6, 3.0)
    assert np.array_equal(gm[0], gm[4])                            # duplicates: equal bits
    for k in (0, 1, 3, 6, 7, 10, 12):                              # alone = inside the bank, bit for bit
        alone, _, _ = run_gpu(d, sigma, traj[k:k + 1], 1.0, t0, 6, 3.0, sep_shape=sep_shape)
        assert np.array_equal(alone[0], gm[k]), k
    # y-jitter breaks the mirror symmetry: no pairs, same answers as the oracle
    jit = np.zeros((T, 2), np.float32)
    jit[:, 1] = 0.3 * np.sin(np.arange(T) / 7.0)
    assert np.all(P.tno_mf_plan_slots(traj, T, t0, jitter_xy=jit)[3] == 0)
    om_j = oracle.snr_map(f, sigma, traj, 1.0, t0, jitter=jit)
    from paper_2209_09848_b200 import MatchedFilter
    with MatchedFilter(0, sep_shape=sep_shape) as mf:
        mj, _ = mf.search(d, sigma, traj, 1.0, t0, jitter_xy=jit)
        torch.cuda.synchronize()
        assert mf.stats()[1] == 1
        assert np.abs(mj.cpu().numpy().astype(np.float64) - om_j).max() <= TOL


@pytest.mark.timeout(180)
def test_many_work_items_per_cta_with_early_flushes():
    """More (tile, batch) work items than SMs, so every CTA walks several items, with trajectories whose
    shift changes within the first frames of an item: the per-entry flush barriers must keep counting
    correctly across item boundaries (a missed wait there once dead-locked the full-size runs)."""
    torch = _torch()
    T, H, W = 12, 1024, 1024
    rng = np.random.default_rng(14)
    f = rng.standard_normal((T, H, W)).astype(np.float32)
    sigma = rng.uniform(0.8, 1.2, T).astype(np.float32)
    traj = np.array([[0.0, 0.45, 0, 0], [0.0, -0.3, 0, 0], [0.0, 0.26, 0, 0.01], [0.0, 0.0, 0, 0],
                     [0.2, 0.5, 0, 0]], np.float32)
    om = oracle.snr_map(f, sigma, traj, 1.0, 0.0)
    gm, gc, stats = run_gpu(torch.from_numpy(f).cuda(), sigma, traj, 1.0, 0.0, 6, 4.5)
    assert stats[1] == 1
    assert np.abs(gm.astype(np.float64) - om).max() <= TOL
    for k in range(traj.shape[0]):
        check_topk_vs_own_map(gc[k], gm[k], k, 6, 4.5)
