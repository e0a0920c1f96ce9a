"""The paper's reproducibility claim: the result does not depend on partition, thread count
or launch configuration. No necsim_sim_params field may change d_events / d_labels / richness."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ns():
    from paper_2108_05815_b200 import necsim
    necsim.lib()
    return necsim


@pytest.fixture(scope="module")
def I():
    from paper_2108_05815_b200 import inputs
    return inputs


def same(a, b):
    return (a["richness"] == b["richness"] and all(np.array_equal(a["events"][f], b["events"][f]) for f in ("loc", "k", "j", "f", "abundance", "time"))
            and np.array_equal(a["labels"], b["labels"]))


@pytest.mark.parametrize("idx", [0, 1, 2, 3, 4])
def test_launch_and_cache_invariance(ns, O, I, idx):
    cfg = I.small_configs()[idx]
    kw = I.scenario_kwargs(cfg)
    ref = O.Scenario(**kw).simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True)
    sc = ns.Scenario(**kw)
    variants = [dict(), dict(block_threads=32, grid_blocks=1), dict(block_threads=64, grid_blocks=7), dict(block_threads=128, grid_blocks=300),
                dict(dedup_log2_slots=4), dict(dedup_log2_slots=10, epoch_events=100), dict(dedup_log2_slots=16, epoch_events=10**9),
                dict(epoch_events=1), dict(tail_threshold=1), dict(tail_threshold=0xFFFFFFFF, epoch_events=3000),
                dict(tail_threshold=500, dedup_log2_slots=8), dict(dedup_probe=1), dict(dedup_probe=4, tail_threshold=1), dict(dedup_probe=2, tail_threshold=0xFFFFFFFF), dict(dedup_probe=7), dict(dedup_probe=6, tail_threshold=1), dict(tail_threshold=0xFFFFFFFF, block_threads=64, grid_blocks=5), dict(dedup=False) if idx in (0, 4) else dict(dedup_log2_slots=12)]
    for v in variants:
        got = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], **v)
        assert same(got, ref), (cfg["name"], v)
    sc.close()


def test_partition_and_merge(ns, O, I):
    """Split the sample into P parts, simulate each separately, merge by unique: same species set (IsolatedIndividuals, L1082-1086)."""
    cfg = I.small_configs()[3]
    kw = I.scenario_kwargs(cfg)
    sc = ns.Scenario(**kw)
    full = sc.simulate(cfg["seed"], cfg["nu"], None)
    n = sc.n_individuals
    rng = np.random.default_rng(0)
    part = rng.integers(0, 3, n)
    keys, labels_keys = set(), {}
    for p in range(3):
        m = (part == p).astype(np.uint8)
        r = sc.simulate(cfg["seed"], cfg["nu"], m)
        ev = r["events"]
        ks = [(int(e["k"]), int(e["f"]), int(e["loc"]), int(e["j"])) for e in ev]
        keys.update(ks)
        for pos, lab in zip(np.flatnonzero(m), r["labels"]):
            labels_keys[int(pos)] = ks[lab]
    merged = sorted(keys)
    fk = [(int(e["k"]), int(e["f"]), int(e["loc"]), int(e["j"])) for e in full["events"]]
    assert merged == fk
    assert all(merged.index(labels_keys[i]) == full["labels"][i] for i in range(0, n, 37))
    sc.close()


@pytest.mark.parametrize("idx", [3, 4])
def test_tail_without_horizon_worst_case(ns, O, I, idx):
    """Guard for the worst case of the one-launch tail: the whole run as ONE tail launch without a horizon
    and a duplicate-culling cache far too small to hold the leaders' entries (16 slots), so that merged lineages hardly ever find
    each other again. The result must still be the oracle's, and the redundant work is bounded by the run without any culling."""
    cfg = I.small_configs()[idx]
    kw = I.scenario_kwargs(cfg)
    ref = O.Scenario(**kw).simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True)
    sc = ns.Scenario(**kw)
    worst = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], tail_threshold=0xFFFFFFFF, dedup_log2_slots=4)
    good = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], tail_threshold=0xFFFFFFFF)
    none = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], tail_threshold=0xFFFFFFFF, dedup=False)
    assert same(worst, ref) and same(good, ref)
    assert worst["stats"]["n_epochs"] == 1 and worst["stats"]["n_tail_epochs"] == 1
    uniq = ref["stats"]["n_events"]                      # the oracle's exact culling: distinct events
    ew, eg, en = worst["stats"]["n_events_raw"], good["stats"]["n_events_raw"], none["stats"]["n_events_raw"]
    print("redundancy over %d distinct events: 16-slot cache %.2f, default cache %.2f, no culling %.2f" % (uniq, ew / uniq, eg / uniq, en / uniq))
    assert uniq <= eg <= ew <= en
    sc.close()
