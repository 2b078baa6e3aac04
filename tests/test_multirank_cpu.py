"""N > 1 host logic of bench.py on CPU: world_size 2, gloo.  The path shards by star with no
data-path collective; what is distributed is the star partition and the
max-over-ranks of the timings.  Also checks that the oracle gives the same trend whether the
stars are processed in one piece or rank by rank (stars are independent)."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from oracle import umi_oracle as orc
    from workloads import lightcurves as lc
    stars = bench.shard_stars(rank, world, 3)
    flux = lc.stars(2, stars)[:, :1500].copy()
    trend = orc.detrend(flux, 51).trend32
    np.save(os.path.join(out_dir, "trend_%d.npy" % rank), trend)
    np.save(os.path.join(out_dir, "stars_%d.npy" % rank), np.array(list(stars)))
    m = bench.max_over_ranks(10.0 + rank, dist)
    dist.barrier()
    np.save(os.path.join(out_dir, "max_%d.npy" % rank), np.array([m]))
    dist.destroy_process_group()


def test_two_ranks_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    from oracle import umi_oracle as orc
    from workloads import lightcurves as lc
    owned = np.concatenate([np.load(tmp_path / ("stars_%d.npy" % r)) for r in range(world)])
    assert sorted(owned.tolist()) == list(range(6))           # disjoint, complete
    whole = orc.detrend(lc.stars(2, range(6))[:, :1500].copy(), 51).trend32
    parts = np.concatenate([np.load(tmp_path / ("trend_%d.npy" % r)) for r in range(world)])
    assert np.array_equal(whole, parts, equal_nan=True)
    for r in range(world):
        assert np.load(tmp_path / ("max_%d.npy" % r))[0] == 11.0  # max over ranks, same on every rank


def test_single_process_helpers():
    import bench
    assert list(bench.shard_stars(0, 1, 4)) == [0, 1, 2, 3]
    assert list(bench.shard_stars(3, 8, 2)) == [6, 7]
    assert bench.max_over_ranks(2.5, None) == 2.5
