"""NEXT-2: isolated partitions + device-side merge give the whole sample's result bit-exactly
(the paper's IsolatedLandscape mode). Ranks are emulated one after another on one GPU; the all-gather
plumbing itself is covered on CPU by tests/test_dist_gloo.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("idx", [1, 3, 4])
@pytest.mark.parametrize("world", [1, 3, 5])
def test_partition_merge_equals_whole(O, idx, world):
    import torch
    from paper_2108_05815_b200 import inputs as I, necsim as ns, dist as D
    cfg = I.small_configs()[idx]
    kw = I.scenario_kwargs(cfg)
    ref = O.Scenario(**kw).simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True)
    sc = ns.Scenario(**kw)
    tabs, labs, masks = [], [], []
    for r in range(world):
        m = D.shard_mask(cfg["mask"], sc.n_individuals, r, world)
        res = sc.simulate_raw(cfg["seed"], cfg["nu"], torch.from_numpy(m).cuda(), int(m.sum()), None)
        t, l = sc.result_tensors(res)
        tabs.append(t.clone()); labs.append(l.to(torch.int64).clone()); masks.append(m)
    offsets = np.cumsum([0] + [t.numel() // 32 for t in tabs])
    merged, dmap = ns.merge_species(torch.cat(tabs))
    ev = merged.cpu().numpy().view(ns.EVENT_DTYPE)
    assert len(ev) == ref["richness"]
    for f in ("loc", "k", "j", "f", "abundance", "time"):
        assert np.array_equal(ev[f], ref["events"][f]), f
    # labels: every rank's lineages, translated through the map, in canonical order of the whole sample
    sampled = np.flatnonzero(np.ones(sc.n_individuals, np.uint8) if cfg["mask"] is None else cfg["mask"])
    glob = np.full(sc.n_individuals, -1, np.int64)
    for r in range(world):
        glob[np.flatnonzero(masks[r])] = dmap[int(offsets[r]) + labs[r]].cpu().numpy()
    assert np.array_equal(glob[sampled], ref["labels"].astype(np.int64))
    # the one-call path with world = 1
    out = D.simulate_partitioned(sc, cfg["seed"], cfg["nu"], cfg["mask"])
    assert out["richness"] == ref["richness"] and np.array_equal(out["labels"].cpu().numpy(), ref["labels"].astype(np.int64))
    sc.close()


def test_partitioned_with_step_cap_marks_unfinished(O):
    """with max_steps some lineages end unfinished (label 0xFFFFFFFF); the translated labels keep them at -1, the others
    agree with the oracle's run under the same cap (dedup off on both sides: per-lineage results are then scheduling-independent)."""
    import torch
    from paper_2108_05815_b200 import inputs as I, necsim as ns, dist as D
    cfg = I.small_configs()[0]
    kw = I.scenario_kwargs(cfg)
    ref = O.Scenario(**kw).simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=False, max_steps=300)
    assert 0 < ref["stats"]["n_unfinished"] < ref["stats"]["n_lineages"]
    sc = ns.Scenario(**kw)
    out = D.simulate_partitioned(sc, cfg["seed"], cfg["nu"], cfg["mask"], params=ns.make_params(dedup=False, max_steps=300))
    lab = out["labels"].cpu().numpy()
    want = ref["labels"].astype(np.int64); want[ref["labels"] == 0xFFFFFFFF] = -1
    assert np.array_equal(lab, want) and out["richness"] == ref["richness"]
    # every lineage unfinished: empty tables, no merge call, all labels -1
    out = D.simulate_partitioned(sc, cfg["seed"], cfg["nu"], cfg["mask"], params=ns.make_params(dedup=False, max_steps=1))
    if out["richness"] == 0:
        assert (out["labels"].cpu().numpy() == -1).all()
    sc.close()
