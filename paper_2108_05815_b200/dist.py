"""Multi-process plumbing for `bench.py --gpus N`: replicas only, no data-path collective.

Every rank simulates an independent replicate (own seed) of the same landscape; the job-level numbers are the
sum of the units processed and the max of the device times over ranks. Works with NCCL (GPU tensors) and with
gloo (CPU tensors; the world-size-2 test in tests/test_dist_gloo.py).
"""
import torch
import torch.distributed as dist


def replica_seed(seed, rank):
    """Seed of rank `rank`'s replicate simulation (distinct u64 per rank, rank 0 keeps the config's seed)."""
    return (int(seed) + int(rank)) & (2**64 - 1)


def aggregate(times_ms, units, device="cpu"):
    """times_ms, units: lists of per-rank floats. Returns (max over ranks of each time, sum over ranks of each unit)."""
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    u = torch.tensor(list(units), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return t.tolist(), u.tolist()


def shard_mask(mask, n_individuals, rank, world):
    """Rank `rank`'s share of the sample: a contiguous range of the sampled individuals in canonical order (cells row-major:
    spatially coherent, the paper's IsolatedLandscape partitioning). Returns a uint8 numpy mask."""
    import numpy as np
    m = np.ones(n_individuals, np.uint8) if mask is None else (np.asarray(mask) != 0).astype(np.uint8)
    idx = np.flatnonzero(m)
    lo, hi = (len(idx) * rank) // world, (len(idx) * (rank + 1)) // world
    out = np.zeros(n_individuals, np.uint8)
    out[idx[lo:hi]] = 1
    return out


def gather_tables(local, record_bytes=32):
    """All-gathers variable-length byte tensors (one species table per rank). Returns (concatenation in rank order,
    per-rank record offsets). The one exchange step of the partitioned path: sizes, then padded tables."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local, [0]
    world = dist.get_world_size()
    n = torch.tensor([local.numel()], dtype=torch.int64, device=local.device)
    sizes = [torch.zeros_like(n) for _ in range(world)]
    dist.all_gather(sizes, n)
    sizes = [int(s.item()) for s in sizes]
    pad = torch.zeros(max(max(sizes), 1), dtype=torch.uint8, device=local.device)
    pad[: local.numel()] = local
    bufs = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(bufs, pad)
    cat = torch.cat([b[:s] for b, s in zip(bufs, sizes)])
    offsets, acc = [], 0
    for s in sizes:
        offsets.append(acc // record_bytes); acc += s
    return cat, offsets


def translate_labels(labels, dmap, offset):
    """Labels of one partition -> ranks in the merged table: dmap[offset + label]. An unfinished lineage (stopped by
    max_steps: label 0xFFFFFFFF, i.e. -1 once widened from the int32 storage) stays -1 instead of indexing a neighbour's record."""
    labels = labels.to(torch.int64)
    unf = (labels < 0) | (labels >= 0xFFFFFFFF)
    if dmap.numel() == 0:
        return torch.full_like(labels, -1)
    out = dmap[offset + torch.where(unf, torch.zeros_like(labels), labels)]
    return torch.where(unf, torch.full_like(out, -1), out)


def simulate_partitioned(scenario, seed, nu, mask=None, rank=0, world=1, params=None):
    """Isolated partitions + merge: this rank simulates its share of the sample with no
    communication, then ONE all-gather of the species tables and a device-side merge (necsim_merge_species) give the table
    of the whole sample. Returns dict(events: CUDA uint8 [S * 32] merged table, labels: CUDA int64 [local lineages] indices
    into it (-1 = unfinished, stopped by max_steps), richness, local: the rank's Result, ms_merge: device time of gather + merge)."""
    from . import necsim as ns
    m = shard_mask(mask, scenario.n_individuals, rank, world)
    if int(m.sum()) == 0:
        local_tab = torch.empty(0, dtype=torch.uint8, device="cuda"); labels = torch.empty(0, dtype=torch.int64, device="cuda"); res = None
    else:
        res = scenario.simulate_raw(seed, nu, torch.from_numpy(m).cuda(), int(m.sum()), params)
        tab, lab = scenario.result_tensors(res)
        local_tab, labels = tab.clone(), lab.to(torch.int64)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    cat, offsets = gather_tables(local_tab)
    if cat.numel() == 0:      # no rank reached a speciation (every lineage unfinished): nothing to merge
        merged, dmap = cat, torch.empty(0, dtype=torch.int64, device=cat.device)
    else:
        merged, dmap = ns.merge_species(cat)
    out_labels = translate_labels(labels, dmap, offsets[rank if len(offsets) > 1 else 0])
    e1.record(); e1.synchronize()
    return dict(events=merged, labels=out_labels, richness=merged.numel() // 32, local=res, ms_merge=e0.elapsed_time(e1))


def throughput(units_total, time_ms_max):
    """Whole-job units per second: everything all ranks processed over the slowest rank's time."""
    return units_total / (time_ms_max * 1e-3)
