"""Multi-GPU path (trajectory sharding, no collective on the data path) exercised with two gloo ranks on the CPU.
The compute stand-in here is the oracle (tests may use it): what is under test is the host logic -- the shard
arithmetic, the Philox trajectory offset, and bench.py's barrier + max-over-ranks timing reduction."""
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1003_1148_b200.sharding import shard_trajectories


def test_shard_arithmetic():
    for T in (0, 1, 5, 256, 257):
        for W in (1, 2, 3, 8):
            seen = []
            for r in range(W):
                off, n = shard_trajectories(T, r, W)
                seen += list(range(off, off + n))
            assert seen == list(range(T))
            sizes = [shard_trajectories(T, r, W)[1] for r in range(W)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_trajectories(4, 2, 2)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, T, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    from oracle import sopo
    from workloads import generators as gen
    import bench
    w = gen.tiny(48, 3)
    off, n = shard_trajectories(T, rank, world)
    o = sopo.from_workload(w, n_traj=n, traj_offset=off)
    o.run(30)
    np.save(os.path.join(out_dir, f"x{rank}.npy"), o.get_coords())
    # the timing reduction bench.py uses: max over ranks; the unit count: sum over ranks
    t = bench.max_over_ranks(float(rank + 1))
    units = bench.sum_over_ranks(float(n))
    np.save(os.path.join(out_dir, f"t{rank}.npy"), np.array([t, units]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_reproduce_the_unsharded_batch(tmp_path):
    T = 5
    mp.spawn(_worker, args=(2, _free_port(), T, str(tmp_path)), nprocs=2, join=True)
    from oracle import sopo
    from workloads import generators as gen
    w = gen.tiny(48, 3)
    ref = sopo.from_workload(w, n_traj=T); ref.run(30)
    got = np.concatenate([np.load(tmp_path / "x0.npy"), np.load(tmp_path / "x1.npy")])
    assert np.array_equal(got, ref.get_coords())
    for r in range(2):
        t, units = np.load(tmp_path / f"t{r}.npy")
        assert t == 2.0 and units == T
