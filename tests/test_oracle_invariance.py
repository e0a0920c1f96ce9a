"""P9 -- the paper's reproducibility claim: the result is independent of how often,
in which order and in which partition lineages are simulated, and of the deduplication (L944)."""
import json
import os
import numpy as np

from paper_2108_05815_b200 import inputs as I

HERE = os.path.dirname(os.path.abspath(__file__))


def run(O, cfg, **kw):
    sc = O.Scenario(**I.scenario_kwargs(cfg))
    return sc, sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], **kw)


def same(a, b):
    return a["richness"] == b["richness"] and (a["events"] == b["events"]).all() and (a["labels"] == b["labels"]).all()


def test_dedup_and_epoch_invariance(O):
    for cfg in I.small_configs():
        sc, ref = run(O, cfg)
        assert same(ref, sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=False))
        for ee in (1000, 37, 10 ** 6):
            assert same(ref, sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True, epoch_events=ee))
        # no-dedup per-lineage terminal events are exactly the labelled events
        nd = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=False, per_lineage=True)
        ev = ref["events"][ref["labels"]]
        for name in ("loc", "k", "j", "f"):
            assert (nd["per_lineage"][name] == ev[name]).all()
        assert nd["steps"].sum() == nd["stats"]["n_events"]


def test_partition_and_merge(O):
    """Split the sample into P parts, simulate each alone (IsolatedIndividuals, L1086), merge by unique event."""
    for cfg in I.small_configs():
        sc, ref = run(O, cfg)
        n_ind = sc.n_individuals
        full = np.ones(n_ind, np.uint8) if cfg["mask"] is None else cfg["mask"].astype(np.uint8)
        sampled = np.flatnonzero(full)
        rng = np.random.default_rng(0)
        part = rng.integers(0, 3, len(sampled))
        merged = {}
        labels_by_ind = {}
        for p in range(3):
            mask = np.zeros(n_ind, np.uint8); mask[sampled[part == p]] = 1
            if mask.sum() == 0: continue
            r = sc.simulate(cfg["seed"], cfg["nu"], mask)
            ev = r["events"]
            for ind, lab in zip(np.flatnonzero(mask), r["labels"]):
                key = (int(ev[lab]["k"]), int(ev[lab]["f"]), int(ev[lab]["loc"]), int(ev[lab]["j"]))
                labels_by_ind[int(ind)] = key; merged[key] = merged.get(key, 0) + 1
        keys = sorted(merged)
        assert len(keys) == ref["richness"]
        rk = [(int(e["k"]), int(e["f"]), int(e["loc"]), int(e["j"])) for e in ref["events"]]
        assert keys == rk
        assert [merged[k] for k in keys] == [int(a) for a in ref["events"]["abundance"]]
        rank = {k: i for i, k in enumerate(keys)}
        assert [rank[labels_by_ind[int(i)]] for i in sampled] == [int(v) for v in ref["labels"]]


def test_subsample_labels_are_consistent(O):
    """A lineage's species does not depend on who else is simulated."""
    cfg = I.small_configs()[3]
    sc, ref = run(O, cfg)
    n_ind = sc.n_individuals
    mask = np.zeros(n_ind, np.uint8); mask[::5] = 1
    sub = sc.simulate(cfg["seed"], cfg["nu"], mask)
    ev_full = ref["events"][ref["labels"][::5]]
    ev_sub = sub["events"][sub["labels"]]
    for name in ("loc", "k", "j", "f"):
        assert (ev_full[name] == ev_sub[name]).all()


def test_seed_and_delta_t_change_the_realisation(O):
    cfg = I.small_configs()[0]
    sc, ref = run(O, cfg)
    other = sc.simulate(cfg["seed"] + 1, cfg["nu"], cfg["mask"])
    assert not (len(other["events"]) == len(ref["events"]) and (other["events"] == ref["events"]).all())
    kw = I.scenario_kwargs(cfg); kw["delta_t"] = 3.0
    r3 = O.Scenario(**kw).simulate(cfg["seed"], cfg["nu"], cfg["mask"])
    assert not (len(r3["events"]) == len(ref["events"]) and (r3["events"] == ref["events"]).all())


def test_step_cap_reports_unfinished(O):
    cfg = I.small_configs()[0]
    sc = O.Scenario(**I.scenario_kwargs(cfg))
    r = sc.simulate(cfg["seed"], cfg["nu"], None, dedup=False, max_steps=10, per_lineage=True)
    assert r["stats"]["n_unfinished"] > 0 and (r["steps"] <= 10).all()
    assert (r["labels"][r["steps"] == 10] == 0xFFFFFFFF).sum() == r["stats"]["n_unfinished"]


def test_small_config_goldens(O):
    """Regression guard: digests written by tests/golden/gen_golden.py (oracle only)."""
    import sys
    sys.path.insert(0, os.path.join(HERE, "golden"))
    from gen_golden import result_digest
    gold = {g["name"]: g for g in json.load(open(os.path.join(HERE, "golden", "small_configs.json")))}
    for cfg in I.small_configs():
        _, r = run(O, cfg)
        g = gold[cfg["name"]]
        assert r["richness"] == g["richness"] and r["stats"]["n_events"] == g["unique_events"]
        assert result_digest(r) == g["digest"]
