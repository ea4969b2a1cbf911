"""Seeded input generators: determinism, shapes, and the recipe of DESIGN.md.  No GPU needed."""
import numpy as np

import tno_synth


def test_configs_match_baseline_json():
    c = tno_synth.CONFIGS
    assert [(c[i].T, c[i].H, c[i].W, c[i].n_traj) for i in range(1, 6)] == [
        (16, 64, 64, 9), (100, 256, 256, 25), (1000, 2048, 2048, 100), (3888, 2048, 2048, 64),
        (1000, 2048, 2048, 1024)]
    assert c[3].evals == 419430400000 and c[5].prf_sigma == 1.2 and not c[5].want_maps
    assert c[1].t0 == 0.0 and c[3].t0 == 500.0 and c[4].t0 == 1944.0


def test_trajectory_grids():
    t3 = tno_synth.trajectories(tno_synth.CONFIGS[3])
    assert t3.dtype == np.float32 and t3.shape == (100, 4)
    assert np.all(t3[:, 2:] == 0) and t3[0, 0] == np.float32(-0.05) and t3[99, 1] == np.float32(0.05)
    assert np.array_equal(t3[:10, 0], np.linspace(-0.05, 0.05, 10).astype(np.float32))   # vx fastest
    t5 = tno_synth.trajectories(tno_synth.CONFIGS[5])
    assert t5.shape == (1024, 4)
    assert sorted({(float(a), float(b)) for a, b in t5[:, 2:]}) == sorted(
        {(0.0, 0.0), (float(np.float32(2e-5)), 0.0), (float(np.float32(-2e-5)), 0.0),
         (0.0, float(np.float32(2e-5)))})
    assert np.all(t5[:256, 2:] == 0)                                                      # acceleration-major


def test_params_and_frames_are_deterministic_and_follow_the_recipe():
    cfg = tno_synth.CONFIGS[2]
    p1, p2 = tno_synth.make_params(cfg), tno_synth.make_params(cfg)
    for a, b in ((p1.sigma_t, p2.sigma_t), (p1.outlier_pos, p2.outlier_pos), (p1.src_x, p2.src_x),
                 (p1.src_amp, p2.src_amp)):
        assert np.array_equal(a, b)
    assert p1.sigma_t.dtype == np.float32 and 0.8 <= p1.sigma_t.min() and p1.sigma_t.max() <= 1.2
    assert p1.outlier_pos.size == round(0.005 * 256 * 256) and p1.hot_pos.size == 0
    assert np.all((p1.src_amp >= 0.5) & (p1.src_amp <= 3.0)) and len(p1.src_k) == 10
    f7a, f7b = tno_synth.frame_numpy(p1, 7), tno_synth.frame_numpy(p2, 7)
    assert np.array_equal(f7a, f7b) and f7a.dtype == np.float32 and f7a.shape == (256, 256)
    assert not np.array_equal(f7a, tno_synth.frame_numpy(p1, 8))
    mask = np.ones(256 * 256, bool)
    mask[p1.outlier_pos] = False
    clean = f7a.reshape(-1)[mask]
    assert abs(clean.std() / p1.sigma_t[7] - 1.0) < 0.02
    assert f7a.reshape(-1)[~mask].std() > 3.0                 # Laplace(5) outliers sit on fixed pixels
    # sources keep their whole track inside the frame
    for k, x, y in zip(p1.src_k, p1.src_x, p1.src_y):
        reach = 0.2 * 50 + 4
        assert reach <= x < 256 - reach and reach <= y < 256 - reach


def test_config1_sources_on_distinct_trajectories_and_sigma_drift():
    p = tno_synth.make_params(tno_synth.CONFIGS[1])
    assert len(set(p.src_k.tolist())) == 2 and np.all(p.src_amp == 3.0)
    small = tno_synth.scaled(tno_synth.CONFIGS[4], T=2000, H=32, W=32)
    ps = tno_synth.make_params(small)
    assert small.t0 == 1000.0 and ps.sigma_t.min() < 0.8 and ps.sigma_t.max() > 1.2   # +-20 % drift
    hot = tno_synth.make_params(tno_synth.scaled(tno_synth.CONFIGS[3], T=4, H=512, W=512))
    assert hot.hot_pos.size == round(1e-4 * 512 * 512)
    f = tno_synth.frame_numpy(hot, 0)
    assert f.reshape(-1)[hot.hot_pos].mean() > 40
