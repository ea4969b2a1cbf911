"""N > 1 host logic on CPU: two gloo ranks shard the path with no data-path collective; only the
max-over-ranks time reduction and a result gather (for the check) cross ranks.  No GPU needed."""
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2209_09848_b200 import multi


def test_shard_trajectories_covers_the_bank_once():
    for n in (1, 7, 9, 64, 100, 1024):
        for world in (1, 2, 3, 8):
            got = []
            for r in range(world):
                lo, hi = multi.shard_trajectories(n, r, world)
                assert 0 <= lo <= hi <= n
                got += list(range(lo, hi))
            assert got == list(range(n))
            sizes = [multi.shard_trajectories(n, r, world) for r in range(world)]
            assert max(h - l for l, h in sizes) - min(h - l for l, h in sizes) <= 1
    with pytest.raises(ValueError):
        multi.shard_trajectories(5, 2, 2)
    assert multi.aggregate_value(1000, 4, 2.0) == 1000 * 4 / 2e-3


def _worker(rank, world, port, out_dir):
    import sys
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import oracle
    import tno_synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = tno_synth.CONFIGS[1]
    # (a) shard by trajectory: ranks share one stack, outputs are disjoint
    p = tno_synth.make_params(cfg)
    f = tno_synth.stack_numpy(p)
    lo, hi = multi.shard_trajectories(cfg.n_traj, rank, world)
    part = oracle.snr_map(f, p.sigma_t, p.traj[lo:hi], cfg.prf_sigma, cfg.t0)
    np.save(os.path.join(out_dir, "part%d.npy" % rank), part)
    # (b) shard by stack: each rank has its own seed
    rc = multi.rank_config(cfg, rank)
    np.save(os.path.join(out_dir, "sig%d.npy" % rank), tno_synth.make_params(rc).sigma_t)
    # timing reduction: max over ranks
    t = multi.max_over_ranks(10.0 + rank)
    assert t == 10.0 + (world - 1)
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks(tmp_path):
    import oracle
    import tno_synth
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    cfg = tno_synth.CONFIGS[1]
    p = tno_synth.make_params(cfg)
    f = tno_synth.stack_numpy(p)
    full = oracle.snr_map(f, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0)
    got = np.concatenate([np.load(tmp_path / "part0.npy"), np.load(tmp_path / "part1.npy")], axis=0)
    assert np.array_equal(got, full)
    assert not np.array_equal(np.load(tmp_path / "sig0.npy"), np.load(tmp_path / "sig1.npy"))
