"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default necsim_sim_params).

(a) whole result against tests/golden/full_configs.json, written by tests/golden/gen_golden.py --full from the oracle
    only: richness, a SHA-256 over every event field and every label (= element-by-element equality), first/last events;
(b) sampled outputs the oracle computes one by one: for a few sampled individuals the oracle traces that single
    lineage alone (no dedup involved) and the GPU's events[labels[i]] must be the speciation event it reaches.
"""
import hashlib
import json
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))
GOLDEN = {0: os.path.join(HERE, "golden", "full_configs.json"),             # exponential event-time sampler
          1: os.path.join(HERE, "golden", "full_configs_poisson.json")}     # Poisson / order statistics (2.7)


def digest(res):
    h = hashlib.sha256()
    for name in ("loc", "k", "j", "f", "abundance"):
        h.update(np.ascontiguousarray(res["events"][name]).tobytes())
    h.update(np.ascontiguousarray(res["events"]["time"]).tobytes())
    h.update(np.ascontiguousarray(res["labels"]).tobytes())
    return h.hexdigest()


def load_golden(sampler):
    if not os.path.exists(GOLDEN[sampler]):
        pytest.skip(os.path.basename(GOLDEN[sampler]) + " not generated")
    return {g["name"]: g for g in json.load(open(GOLDEN[sampler]))}


@pytest.mark.parametrize("sampler", [0, 1])
@pytest.mark.parametrize("idx", range(5))
def test_full_config_matches_oracle(O, idx, sampler):
    golden = load_golden(sampler)
    from paper_2108_05815_b200 import inputs as I, necsim as ns
    cfg = [I.c1_nonspatial, I.c2_implicit, I.c3_matrix, I.c4_gaussian, I.c5_stress][idx]()
    if cfg["name"] not in golden:
        pytest.skip("no golden record for " + cfg["name"])
    g = golden[cfg["name"]]
    kw = dict(I.scenario_kwargs(cfg), sampler=sampler)
    sc = ns.Scenario(**kw)
    got = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"])
    assert len(got["labels"]) == g["n_sampled"]
    assert got["richness"] == g["richness"]
    ev = got["events"]
    rows = lambda a: [[int(e["loc"]), int(e["k"]), int(e["j"]), int(e["f"]), int(e["abundance"])] for e in a]
    assert rows(ev[:5]) == g["first_events"] and rows(ev[-5:]) == g["last_events"]
    assert [int(v) for v in got["labels"][:16]] == g["labels_head"]
    assert digest(got) == g["digest"]
    # properties that hold at any size
    assert int(ev["abundance"].sum()) == g["n_sampled"] and (ev["abundance"] > 0).all()
    key = np.stack([ev["k"].astype(np.uint64), ev["f"], ev["loc"].astype(np.uint64), ev["j"].astype(np.uint64)], axis=1)
    assert all(tuple(key[i]) < tuple(key[i + 1]) for i in range(len(key) - 1))
    assert got["stats"]["n_events_raw"] >= g["unique_events"]
    # (b) single lineages, one by one
    n_ind = sc.n_individuals
    sampled = np.arange(n_ind) if cfg["mask"] is None else np.flatnonzero(cfg["mask"])
    rng = np.random.default_rng(idx)
    osc = O.Scenario(**kw)
    for pos in rng.choice(len(sampled), 3, replace=False):
        m = np.zeros(n_ind, np.uint8); m[sampled[pos]] = 1
        one = osc.simulate(cfg["seed"], cfg["nu"], m, dedup=False)
        e, mine = one["events"][0], ev[got["labels"][pos]]
        assert (int(e["loc"]), int(e["k"]), int(e["j"]), int(e["f"])) == (int(mine["loc"]), int(mine["k"]), int(mine["j"]), int(mine["f"]))
        assert e["time"] == mine["time"]
    sc.close()


def test_bigdeme_full_size_matches_oracle(O):
    """SURVEY NEXT-4 workload (bench.py --config c6) at full size against tests/golden/full_config_c6.json (oracle only)."""
    from paper_2108_05815_b200 import inputs as I, necsim as ns
    f = os.path.join(HERE, "golden", "full_config_c6.json")
    if not os.path.exists(f):
        pytest.skip("full_config_c6.json not generated")
    g = json.load(open(f))[0]
    cfg = I.c6_bigdeme()
    assert g["name"] == cfg["name"]
    sc = ns.Scenario(**I.scenario_kwargs(cfg))
    got = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"])
    assert got["richness"] == g["richness"] and len(got["labels"]) == g["n_sampled"]
    assert [int(v) for v in got["labels"][:16]] == g["labels_head"]
    assert digest(got) == g["digest"]
    assert got["stats"]["n_events_raw"] >= g["unique_events"]
    sc.close()


def test_habitat_loss_full_size_matches_oracle(O):
    """Temporally varying habitat at full size: the C5 landscape after a habitat loss
    (bench.py --config c7) against tests/golden/full_config_c7.json (oracle only)."""
    from paper_2108_05815_b200 import inputs as I, necsim as ns
    f = os.path.join(HERE, "golden", "full_config_c7.json")
    if not os.path.exists(f):
        pytest.skip("full_config_c7.json not generated")
    g = json.load(open(f))[0]
    cfg = I.c7_habitat_loss()
    assert g["name"] == cfg["name"]
    sc = ns.Scenario(**I.scenario_kwargs(cfg))
    got = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"])
    assert got["richness"] == g["richness"] and len(got["labels"]) == g["n_sampled"]
    assert [int(v) for v in got["labels"][:16]] == g["labels_head"]
    rows = lambda a: [[int(e["loc"]), int(e["k"]), int(e["j"]), int(e["f"]), int(e["abundance"])] for e in a]
    assert rows(got["events"][:5]) == g["first_events"] and rows(got["events"][-5:]) == g["last_events"]
    assert digest(got) == g["digest"]
    assert got["stats"]["n_events_raw"] >= g["unique_events"]
    sc.close()
