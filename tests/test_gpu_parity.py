"""GPU parity of the whole hot path (S0-S6) against the CPU oracle, through the C-ABI: bit-exact species table,
richness, labels and abundances; event times identical (tolerance stated by north_star: 1e-12 relative; both sides
evaluate ((double)k + f*2^-48)*delta_t with the same IEEE operations, so we assert equality and report the bound).
With dedup off, also the per-lineage terminal record and step count."""
import json
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def ns():
    from paper_2108_05815_b200 import necsim
    necsim.lib()
    return necsim


@pytest.fixture(scope="module")
def I():
    from paper_2108_05815_b200 import inputs
    return inputs


def assert_same_result(got, ref, name=""):
    assert got["richness"] == ref["richness"], (name, got["richness"], ref["richness"])
    for f in ("loc", "k", "j", "f", "abundance"):
        assert np.array_equal(got["events"][f], ref["events"][f]), (name, f)
    t_g, t_r = got["events"]["time"], ref["events"]["time"]
    assert np.all(np.abs(t_g - t_r) <= 1e-12 * np.abs(t_r)), name
    assert np.array_equal(t_g, t_r), name
    assert np.array_equal(got["labels"], ref["labels"]), name


KERNELS = {"per_thread": 1, "tail": 0xFFFFFFFF}      # tail_threshold: which simulate kernel runs every epoch


@pytest.mark.parametrize("kernel", sorted(KERNELS))
@pytest.mark.parametrize("idx", range(5))
def test_small_configs_dedup_on(ns, O, I, idx, kernel):
    cfg = I.small_configs()[idx]
    kw = I.scenario_kwargs(cfg)
    ref = O.Scenario(**kw).simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True)
    sc = ns.Scenario(**kw)
    got = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], tail_threshold=KERNELS[kernel])
    assert_same_result(got, ref, cfg["name"])
    assert (got["stats"]["n_tail_epochs"] == got["stats"]["n_epochs"]) == (kernel == "tail")
    golden = json.load(open(os.path.join(HERE, "golden", "small_configs.json")))[idx]     # written by the oracle only
    assert golden["name"] == cfg["name"] and golden["richness"] == got["richness"]
    assert golden["labels_head"] == [int(v) for v in got["labels"][:16]]
    # every unique event is executed at least once; raw >= unique
    assert got["stats"]["n_events_raw"] >= ref["stats"]["n_events"]
    sc.close()


@pytest.mark.parametrize("kernel", sorted(KERNELS))
@pytest.mark.parametrize("idx", range(5))
def test_small_configs_dedup_off_per_lineage(ns, O, I, idx, kernel):
    cfg = I.small_configs()[idx]
    kw = I.scenario_kwargs(cfg)
    nu = max(cfg["nu"], 5e-3)                      # no dedup: n/nu events
    ref = O.Scenario(**kw).simulate(cfg["seed"], nu, cfg["mask"], dedup=False, per_lineage=True)
    sc = ns.Scenario(**kw)
    got = sc.simulate(cfg["seed"], nu, cfg["mask"], per_lineage=True, dedup=False, tail_threshold=KERNELS[kernel])
    assert_same_result(got, ref, cfg["name"])
    for f in ("loc", "k", "j", "f"):
        assert np.array_equal(got["per_lineage"][f], ref["per_lineage"][f]), (cfg["name"], f)
    assert np.array_equal(got["steps"], ref["steps"])
    assert (got["state"] == 1).all()
    assert got["stats"]["n_events_raw"] == ref["stats"]["n_events"] == int(ref["steps"].sum())
    sc.close()


@pytest.mark.parametrize("kernel", sorted(KERNELS))
@pytest.mark.parametrize("idx", [0, 3])
def test_step_cap_mode(ns, O, I, idx, kernel):
    """MODE-T workload: dedup off, every lineage advanced at most max_steps events."""
    cfg = I.small_configs()[idx]
    kw = I.scenario_kwargs(cfg)
    ref = O.Scenario(**kw).simulate(cfg["seed"], 1e-3, cfg["mask"], dedup=False, max_steps=100, per_lineage=True)
    sc = ns.Scenario(**kw)
    got = sc.simulate(cfg["seed"], 1e-3, cfg["mask"], per_lineage=True, dedup=False, max_steps=100, tail_threshold=KERNELS[kernel])
    assert_same_result(got, ref, cfg["name"])
    assert got["stats"]["n_unfinished"] == ref["stats"]["n_unfinished"] > 0
    for f in ("loc", "k", "j", "f"):
        assert np.array_equal(got["per_lineage"][f], ref["per_lineage"][f]), (cfg["name"], f)
    assert np.array_equal(got["steps"], ref["steps"])
    sc.close()


def test_edge_cases(ns, O, I):
    # a single individual; nu = 1 (everyone speciates at the first event); tiny landscapes
    for J, nu in ((1, 0.5), (2, 1.0), (33, 1.0), (5, 0.25)):
        cfg = I.c1_nonspatial(J=J, nu=nu, seed=3)
        kw = I.scenario_kwargs(cfg)
        ref = O.Scenario(**kw).simulate(3, nu, None, dedup=True)
        sc = ns.Scenario(**kw)
        assert_same_result(sc.simulate(3, nu, None), ref, "J=%d" % J)
        sc.close()
    # a mask selecting one individual, and the last individual only
    cfg = I.small_configs()[3]
    kw = I.scenario_kwargs(cfg)
    o = O.Scenario(**kw); sc = ns.Scenario(**kw)
    for pos in (0, sc.n_individuals - 1, 4097 % sc.n_individuals):
        m = np.zeros(sc.n_individuals, np.uint8); m[pos] = 1
        assert_same_result(sc.simulate(5, 1e-2, m), o.simulate(5, 1e-2, m, dedup=True), "single@%d" % pos)
    # errors: empty mask, nu out of range, nu = 0 without a step cap
    with pytest.raises(ns.NecsimError):
        sc.simulate(5, 1e-2, np.zeros(sc.n_individuals, np.uint8))
    with pytest.raises(ns.NecsimError):
        sc.simulate(5, 1.5, None)
    with pytest.raises(ns.NecsimError):
        sc.simulate(5, 0.0, None)
    sc.close()
    with pytest.raises(ns.NecsimError):
        ns.Scenario(I.EXPLICIT_GAUSSIAN, width=8, height=8, uniform_deme=1, sigma=2.0)      # 10*sigma >= width
    with pytest.raises(ns.NecsimError):
        ns.Scenario(I.NONSPATIAL, uniform_deme=0)


def test_host_entry_point_matches(ns, O, I):
    """necsim_simulate_host (host mask in, host events/labels out) gives the same answer."""
    import torch
    cfg = I.small_configs()[4]
    kw = I.scenario_kwargs(cfg)
    ref = O.Scenario(**kw).simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True)
    sc = ns.Scenario(**kw)
    n = int(np.count_nonzero(cfg["mask"]))
    h_mask = torch.from_numpy(np.ascontiguousarray(cfg["mask"])).pin_memory().numpy()
    h_events = torch.empty(n * 32, dtype=torch.uint8).pin_memory().numpy().view(ns.EVENT_DTYPE)
    h_labels = torch.empty(n, dtype=torch.int32).pin_memory().numpy().view(np.uint32)
    res = sc.simulate_host_raw(cfg["seed"], cfg["nu"], h_mask, n, None, h_events, h_labels)
    got = dict(richness=int(res.richness), events=h_events[: res.richness], labels=h_labels[: res.n_lineages])
    assert_same_result(got, ref, cfg["name"])
    sc.close()
