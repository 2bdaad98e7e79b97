"""world_size-2 gloo tests (CPU) of the multi-GPU host logic: contiguous seed sharding, ragged reward
all-gather, max-over-ranks timing, and that every rank ends with the same selection."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import rollout
from paper_2606_19004_b200 import sharding


def test_shard_range_partitions_every_unit_once():
    for n in (0, 1, 5, 16, 17, 256):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                lo, hi = sharding.shard_range(n, r, world)
                assert 0 <= lo <= hi <= n
                seen += list(range(lo, hi))
            assert seen == list(range(n))
            sizes = sharding.shard_sizes(n, world)
            assert max(sizes) - min(sizes) <= 1
    # unit b lives on rank floor(b * world / n)
    lo, hi = sharding.shard_range(16, 1, 2)
    assert (lo, hi) == (8, 16) and all(b * 2 // 16 == 1 for b in range(lo, hi))


def _fake_reward(seed: int) -> float:
    return float(np.sin(seed * 12.9898) * 43758.5453 % 1.0)


def _worker(rank, world, port, n_units, k_select, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lo, hi = sharding.shard_range(n_units, rank, world)
        local = torch.tensor([_fake_reward(s) for s in range(lo, hi)], dtype=torch.float32)
        full = sharding.gather_rewards(local, n_units)
        sel = rollout.select_seeds(full.numpy().astype(np.float64)[None, :], k_select)
        slow = sharding.max_over_ranks(10.0 + rank)
        q.put((rank, full.tolist(), sel["top"].tolist(), sel["bottom"].tolist(), float(sel["std"][0]), slow))
    finally:
        dist.destroy_process_group()


def test_shard_prompt_index_cuts_through_groups():
    """explore_shard runs its slice as one-seed prompt groups: sequence b keeps the text of prompt b // K."""
    P, K, world = 3, 5, 4
    seen = []
    for r in range(world):
        lo, hi = sharding.shard_range(P * K, r, world)
        idx = sharding.shard_prompt_index(lo, hi, K)
        assert len(idx) == hi - lo and all(0 <= p < P for p in idx)
        seen += idx
    assert seen == [b // K for b in range(P * K)]
    assert sharding.shard_prompt_index(4, 6, 5) == [0, 1]              # a shard that straddles two prompt groups
    assert sharding.shard_prompt_index(7, 7, 5) == []


@pytest.mark.parametrize("n_units", [16, 17])
def test_two_rank_gather_and_selection(n_units):
    world, port = 2, 29500 + (os.getpid() % 2000) + n_units
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_units, 4, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want = [float(np.float32(_fake_reward(s))) for s in range(n_units)]
    ref = rollout.select_seeds(np.asarray([want], dtype=np.float64), 4)
    for rank, full, top, bottom, std, slow in results:
        assert full == want                                # ragged shards reassembled in order
        assert top == ref["top"].tolist() and bottom == ref["bottom"].tolist()
        assert abs(std - ref["std"][0]) < 1e-12
        assert slow == 11.0                                # max over ranks
