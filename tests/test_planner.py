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


# ---- slots: mirror pairs (tno_mf_plan_slots) ------------------------------------------------------
from paper_2209_09848_b200 import tno_mf_plan_slots  # noqa: E402


def _check_slots(traj, T, t0, ns=5, sym=True, **kw):
    n, batch, slot, member = tno_mf_plan_slots(traj, T, t0, ns, sym, **kw)
    assert np.all(batch >= 0) and np.all(batch < n) and np.all(slot >= 0) and np.all(slot < ns)
    assert set(member.tolist()) <= {0, 1}
    seen = set(zip(batch.tolist(), slot.tolist(), member.tolist()))
    assert len(seen) == len(traj), "every trajectory owns exactly one (batch, slot, member)"
    for b in range(n):
        ks = np.nonzero(batch == b)[0]
        assert len({(float(traj[k, 0]), float(traj[k, 2])) for k in ks}) == 1, "one x-motion per batch"
        assert sorted(set(slot[ks].tolist())) == list(range(len(set(slot[ks].tolist())))), "slots 0 .. n-1"
        for s in set(slot[ks].tolist()):
            mem = ks[slot[ks] == s]
            if len(mem) == 2:           # a pair: exact mirror images in y, sharing the x-motion
                p, q = (mem[0], mem[1]) if member[mem[0]] == 0 else (mem[1], mem[0])
                assert member[p] == 0 and member[q] == 1
                assert traj[p, 1] == -traj[q, 1] and traj[p, 3] == -traj[q, 3]
                assert traj[p, 1] > 0 or (traj[p, 1] == 0 and traj[p, 3] >= 0)
    return n, batch, slot, member


def _n_pairs(batch, slot):
    _, counts = np.unique(np.stack([batch, slot], 1), axis=0, return_counts=True)
    assert counts.max() <= 2
    return int(np.count_nonzero(counts == 2))


def test_slots_of_the_config_banks():
    """The velocity grids of the five configs are symmetric about zero: every vy < 0 pairs with its mirror image."""
    for idx, batches, pairs in ((1, 3, 3), (2, 5, 10), (3, 10, 50), (4, 8, 32)):
        cfg = tno_synth.CONFIGS[idx]
        traj = tno_synth.trajectories(cfg)
        n, batch, slot, member = _check_slots(traj, cfg.T, cfg.t0)
        assert n == batches
        assert _n_pairs(batch, slot) == pairs
    # config 5: ay = +2e-5 has no mirror image in the bank -> 256 single slots (the 128 with vy < 0 are lone
    # minus members), (1024 - 256) / 2 pairs
    cfg = tno_synth.CONFIGS[5]
    traj = tno_synth.trajectories(cfg)
    n, batch, slot, member = _check_slots(traj, cfg.T, cfg.t0)
    assert _n_pairs(batch, slot) == 384 and int(np.count_nonzero(member == 1)) == 384 + 128
    assert n == 16 * 5 + 32 * 2            # ax = 0: 8 pairs + 16 singles = 24 slots; ax != 0: 8 pairs


def test_no_pairs_without_symmetry_with_ties_or_with_y_jitter():
    traj = np.array([[0.1, v, 0, 0] for v in (-0.3, -0.1, 0.0, 0.1, 0.3)], dtype=np.float32)
    assert np.count_nonzero(_check_slots(traj, 40, 20.0)[3] == 1) == 2
    assert np.count_nonzero(_check_slots(traj, 40, 20.0, sym=False)[3] == 1) == 0
    jit = np.zeros((40, 2), np.float32)
    jit[:, 0] = 0.3                                             # jitter in x only: still pairs
    assert np.count_nonzero(_check_slots(traj, 40, 20.0, jitter_xy=jit)[3] == 1) == 2
    jit[7, 1] = 0.01                                            # any jitter in y breaks the mirror symmetry
    assert np.count_nonzero(_check_slots(traj, 40, 20.0, jitter_xy=jit)[3] == 1) == 0
    # exact half-pixel ties (v = +-0.5 at odd dt): floor(-d + 1/2) != -floor(d + 1/2), so +-0.5 must not pair,
    # while +-0.3 (never exactly on a tie) still do
    tie = np.array([[0, 0.5, 0, 0], [0, -0.5, 0, 0], [0, 0.3, 0, 0], [0, -0.3, 0, 0]], dtype=np.float32)
    n, batch, slot, member = _check_slots(tie, 10, 0.0)
    assert member[0] == 0 and member[1] == 0 and slot[0] != slot[1]
    assert member[2] == 0 and member[3] == 1 and slot[2] == slot[3]
    # irregular frame times keep the symmetry (d is odd in (v, a) for any dt)
    times = np.cumsum(np.random.default_rng(0).uniform(0.5, 1.5, 40)).astype(np.float32)
    assert np.count_nonzero(_check_slots(traj, 40, 20.0, frame_times=times)[3] == 1) == 2


def test_duplicates_and_lonely_mirror_images():
    traj = np.array([[0.1, 0.2, 0, 0], [0.1, 0.2, 0, 0], [0.1, -0.2, 0, 0], [0.2, -0.4, 0, 1e-4], [0.1, 0.0, 0, 0],
                     [0.1, 0.0, 0, 0]], dtype=np.float32)
    n, batch, slot, member = _check_slots(traj, 30, 15.0)
    assert n == 2
    assert member.tolist() == [0, 0, 1, 1, 0, 0]                # a lone negative motion is the minus member
    assert slot[0] != slot[1] and slot[2] in (slot[0], slot[1])  # the duplicate gets a slot of its own
    assert slot[4] != slot[5]
    with pytest.raises(TnoMfError):
        tno_mf_plan_slots(traj, 30, float("nan"))
    with pytest.raises(TnoMfError):
        tno_mf_plan_slots(traj, 30, 0.0, 17)
