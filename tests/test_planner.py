"""Host planner (tno_mf_plan): trajectories are grouped into batches that share one x-motion and
whose integer y-shifts stay within the allowed spread.  Checked against an independent
computation of the shifts.  No GPU needed."""
import math
from fractions import Fraction

import numpy as np
import pytest

import tno_synth
from paper_2209_09848_b200 import TnoMfError, tno_mf_plan


def _shift(v, a, t, t0):
    dt = Fraction(t) - Fraction(float(t0))
    d = Fraction(float(np.float32(v))) * dt + Fraction(float(np.float32(a))) * dt * dt
    return math.floor(d + Fraction(1, 2))


def _check(traj, T, t0, nb, spread):
    n, batch, slot = tno_mf_plan(traj, T, t0, nb, spread)
    assert n >= 1 and np.all(batch >= 0) and np.all(batch < n) and np.all(slot >= 0) and np.all(slot < nb)
    seen = set(zip(batch.tolist(), slot.tolist()))
    assert len(seen) == len(traj), "every trajectory owns exactly one (batch, slot)"
    ts = sorted(set([0, T - 1, T // 2, T // 3, (2 * T) // 3] + list(range(0, T, max(1, T // 37)))))
    for b in range(n):
        ks = np.nonzero(batch == b)[0]
        assert 1 <= len(ks) <= nb
        assert len({(float(traj[k, 0]), float(traj[k, 2])) for k in ks}) == 1, "one x-motion per batch"
        assert sorted(slot[ks].tolist()) == list(range(len(ks)))
        for t in ts:
            s = [_shift(traj[k, 1], traj[k, 3], t, t0) for k in ks]
            assert max(s) - min(s) <= spread
    return n


@pytest.mark.parametrize("idx,nb,spread,expect", [
    (1, 8, 60, 3), (1, 10, 60, 3), (2, 8, 60, 5), (3, 10, 60, 10), (3, 8, 60, 20),
    (4, 8, 60, 8), (5, 8, 60, 128),
])
def test_config_banks(idx, nb, spread, expect):
    cfg = tno_synth.CONFIGS[idx]
    traj = tno_synth.trajectories(cfg)
    assert _check(traj, cfg.T, cfg.t0, nb, spread) == expect


def test_spread_limit_splits_batches_and_singletons_always_fit():
    traj = np.array([[0.0, v, 0, 0] for v in np.linspace(-1, 1, 9)], dtype=np.float32)
    assert _check(traj, 200, 100.0, 8, 1000) == 2          # 8 + 1
    n_tight = _check(traj, 200, 100.0, 8, 30)              # neighbours drift 25 px apart at the ends
    assert n_tight >= 5
    assert _check(traj, 200, 100.0, 8, 0) == 9             # spread 0: every trajectory alone


def test_unshared_motions_and_duplicates():
    rng = np.random.default_rng(0)
    traj = rng.uniform(-0.3, 0.3, size=(13, 4)).astype(np.float32)
    traj[:, 2:] *= 1e-3
    assert _check(traj, 50, 25.0, 8, 60) == 13             # no two share an x-motion
    dup = np.repeat(np.array([[0.1, 0.2, 0, 0]], np.float32), 5, axis=0)
    assert _check(dup, 50, 0.0, 8, 60) == 1                # duplicates are separate entries


def test_bad_arguments():
    traj = np.zeros((2, 4), np.float32)
    for args in ((0, 0.0, 8, 60), (10, 0.0, 0, 60), (10, 0.0, 17, 60), (10, 0.0, 8, -1),
                 (10, float("nan"), 8, 60)):
        with pytest.raises(TnoMfError):
            tno_mf_plan(traj, *args)
    traj[1, 0] = np.inf
    with pytest.raises(TnoMfError):
        tno_mf_plan(traj, 10, 0.0, 8, 60)
    with pytest.raises(TnoMfError):                          # displacement beyond 1e9 px
        tno_mf_plan(np.array([[3e8, 0, 0, 0]], np.float32), 100, 0.0, 8, 60)


def test_unlimited_spread_splits_evenly():
    """max_spread >= 2^30 is what the search itself uses: no spread limit, each x-motion is split into
    the fewest batches, of sizes that differ by at most one."""
    unlimited = 1 << 30
    traj = np.array([[0.1, v, 0, 0] for v in np.linspace(-3, 3, 23)] +
                    [[0.2, v, 0, 0] for v in np.linspace(-1, 1, 10)] + [[0.3, 0, 0, 0]], dtype=np.float32)
    n, batch, slot = tno_mf_plan(traj, 100, 50.0, 10, unlimited)
    assert n == 3 + 1 + 1
    sizes = sorted(np.bincount(batch).tolist())
    assert sizes == [1, 7, 8, 8, 10]
    for b in range(n):
        ks = np.nonzero(batch == b)[0]
        assert len({float(traj[k, 0]) for k in ks}) == 1
        assert sorted(slot[ks].tolist()) == list(range(len(ks)))
    for idx, nb, expect in ((3, 10, 10), (5, 8, 128), (5, 10, 128), (4, 8, 8)):
        cfg = tno_synth.CONFIGS[idx]
        assert tno_mf_plan(tno_synth.trajectories(cfg), cfg.T, cfg.t0, nb, unlimited)[0] == expect
