"""GPU parity of the full event stream: the device-sorted, device-deduplicated stream of every executed
event equals the oracle's, field by field, for both simulate kernels and both event-time samplers; and recording does
not change the species result."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
KERNELS = {"per_thread": 1, "tail": 0xFFFFFFFF}


@pytest.mark.parametrize("sampler", [0, 1])
@pytest.mark.parametrize("kernel", sorted(KERNELS))
def test_stream_matches_oracle(O, kernel, sampler):
    from paper_2108_05815_b200 import inputs as I, necsim as ns
    for cfg in I.small_configs():
        kw = dict(I.scenario_kwargs(cfg), sampler=sampler)
        ref = O.Scenario(**kw).simulate_stream(cfg["seed"], cfg["nu"], cfg["mask"])
        sc = ns.Scenario(**kw)
        # stream_sort_bytes = 1: most records agree on the radix-sorted key prefix, so the order comes from the tie pass
        for knobs in (dict(), dict(event_ring_capacity=60_000, epoch_events=3000, dedup_log2_slots=8), dict(dedup=False, event_ring_capacity=2**22),
                      dict(stream_sort_bytes=1), dict(stream_sort_bytes=5, event_ring_capacity=60_000, epoch_events=3000)):
            if knobs.get("dedup") is False and cfg["nu"] < 1e-3:
                continue
            got = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], record_events=True, event_stream_capacity=2**21,
                              tail_threshold=KERNELS[kernel], **knobs)
            assert got["richness"] == ref["richness"] and np.array_equal(got["labels"], ref["labels"])
            assert len(got["stream"]) == len(ref["stream"]) == got["stats"]["n_stream_events"], (cfg["name"], knobs)
            for f in ("loc", "k", "j", "f", "loc2"):
                assert np.array_equal(got["stream"][f], ref["stream"][f]), (cfg["name"], knobs, f)
        sc.close()


def test_stream_capacity_errors(O):
    from paper_2108_05815_b200 import inputs as I, necsim as ns
    cfg = I.small_configs()[3]
    sc = ns.Scenario(**I.scenario_kwargs(cfg))
    with pytest.raises(ns.NecsimError):
        sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], record_events=True, event_stream_capacity=100)
    with pytest.raises(ns.NecsimError):
        sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], record_events=True, event_ring_capacity=64)
    with pytest.raises(ns.NecsimError):
        sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], record_events=True, stream_sort_bytes=6)
    out = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"])        # the handle still works
    assert out["richness"] > 0
    sc.close()


def test_full_size_stream_counts_match_the_oracle():
    """At full size the stream holds exactly the oracle's number of distinct events (tests/golden/full_configs.json), in time
    order, with one speciation record per species."""
    import json, os
    from paper_2108_05815_b200 import inputs as I, necsim as ns
    golden = {g["name"]: g for g in json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "full_configs.json")))}
    for cfg, ring, cap in ((I.c4_gaussian(), 2**24, 2**24), (I.c2_implicit(), 2**24, 2**26)):
        sc = ns.Scenario(**I.scenario_kwargs(cfg))
        got = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], record_events=True, event_ring_capacity=ring, event_stream_capacity=cap)
        g = golden[cfg["name"]]
        st = got["stream"]
        assert len(st) == g["unique_events"] and got["richness"] == g["richness"]
        assert int((st["loc2"] == 0xFFFFFFFF).sum()) == g["richness"]
        t = st["k"].astype(np.float64) + st["f"].astype(np.float64) / 2.0**48
        assert np.all(np.diff(t) >= 0)
        sc.close()
