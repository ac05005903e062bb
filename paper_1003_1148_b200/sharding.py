"""Multi-GPU: the path shards only across trajectories (PAPER.md:292 many-runs-per-GPU; :310 several GPUs, one run
each).  No collective is involved: rank r simulates a contiguous slice of the batch, and the Philox trajectory
word (`traj_offset`) makes the union of the shards bit-identical to the unsharded batch."""
from __future__ import annotations


def shard_trajectories(n_traj_total: int, rank: int, world_size: int):
    """-> (traj_offset, n_local): contiguous slices, sizes differing by at most one, every trajectory owned once."""
    if not (0 <= rank < world_size) or n_traj_total < 0:
        raise ValueError("bad rank / world_size / n_traj_total")
    base, extra = divmod(n_traj_total, world_size)
    n_local = base + (1 if rank < extra else 0)
    offset = rank * base + min(rank, extra)
    return offset, n_local
