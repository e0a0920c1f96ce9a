"""World-size-2 gloo test (CPU) of the N>1 host logic bench.py uses: replica seeds, sum of units, max of times."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2108_05815_b200 import dist as D
    seed = D.replica_seed(42, rank)
    times, units = D.aggregate([10.0 + 5.0 * rank, 3.0 - rank], [1000.0 * (rank + 1), 7.0])
    # the exchange step of the partitioned path: variable-length tables, rank order, record offsets
    tab = torch.full((32 * (rank + 2),), rank + 1, dtype=torch.uint8)
    cat, offsets = D.gather_tables(tab)
    assert offsets == [0, 2] and cat.numel() == 32 * 5 and bool((cat[:64] == 1).all()) and bool((cat[64:] == 2).all())
    # uneven and EMPTY shards: rank 1 contributes no species table at all
    tab2 = torch.full((32 * 3,), 7, dtype=torch.uint8) if rank == 0 else torch.empty(0, dtype=torch.uint8)
    cat2, off2 = D.gather_tables(tab2)
    assert off2 == [0, 3] and cat2.numel() == 96 and bool((cat2 == 7).all())
    # label translation of this rank's lineages through a merged map (the step after the gather)
    dmap = torch.arange(10, 15, dtype=torch.int64)                      # merged rank of each of the 5 gathered records
    lab = torch.tensor([0, 1, -1] if rank == 0 else [2, 0, -1], dtype=torch.int64)
    assert D.translate_labels(lab, dmap, offsets[rank]).tolist() == ([10, 11, -1] if rank == 0 else [14, 12, -1])
    out[rank] = (seed, times, units, D.throughput(units[0], times[0]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation():
    world, port = 2, _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    assert out[0][0] == 42 and out[1][0] == 43
    for r in range(world):
        _, times, units, thr = out[r]
        assert times == [15.0, 3.0]                 # max over ranks
        assert units == [3000.0, 14.0]              # sum over ranks
        assert abs(thr - 3000.0 / 0.015) < 1e-6


def test_shard_mask_partitions_the_sample():
    import numpy as np
    from paper_2108_05815_b200 import dist as D
    rng = np.random.default_rng(0)
    mask = (rng.random(1000) < 0.3).astype(np.uint8)
    for world in (1, 2, 7):
        parts = [D.shard_mask(mask, 1000, r, world) for r in range(world)]
        assert np.array_equal(np.sum(parts, axis=0), mask)                     # disjoint cover of the sample
        firsts = [np.flatnonzero(p)[0] for p in parts if p.any()]
        assert firsts == sorted(firsts)                                        # contiguous ranges in canonical order
        assert max(int(p.sum()) for p in parts) - min(int(p.sum()) for p in parts) <= 1
    assert np.array_equal(D.shard_mask(None, 10, 1, 2), np.array([0] * 5 + [1] * 5, np.uint8))


def test_single_process_is_identity():
    from paper_2108_05815_b200 import dist as D
    assert D.aggregate([1.5], [2.0]) == ([1.5], [2.0])
    assert D.replica_seed(2**64 - 1, 1) == 0


def test_translate_labels_keeps_unfinished_and_handles_empty_tables():
    """a lineage stopped by max_steps (label 0xFFFFFFFF -> -1 in int64) must not index a neighbour's record."""
    from paper_2108_05815_b200 import dist as D
    dmap = torch.tensor([5, 6, 7, 8, 9], dtype=torch.int64)
    lab = torch.tensor([0, -1, 1, 0xFFFFFFFF], dtype=torch.int64)
    assert D.translate_labels(lab, dmap, 2).tolist() == [7, -1, 8, -1]
    assert D.translate_labels(lab, dmap, 0).tolist() == [5, -1, 6, -1]          # rank 0: no negative wrap to the last record
    assert D.translate_labels(torch.tensor([-1, -1]), torch.empty(0, dtype=torch.int64), 0).tolist() == [-1, -1]
    assert D.translate_labels(torch.empty(0, dtype=torch.int64), dmap, 3).numel() == 0
