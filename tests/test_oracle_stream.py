"""Pins of the oracle's full event stream (PAPER.md 6.2 L813-906, 7.1.3 L958-967): what the stream must
satisfy whatever the implementation -- one record per distinct executed event, one speciation record per species, time
order, and closure: the lineage that dispersed to loc2 at time t executes loc2's next event after t, so that event is in the
stream too (checked by brute force with the event-time search)."""
import numpy as np


def test_stream_identities_and_closure(O):
    from paper_2108_05815_b200 import inputs as I
    for idx in (0, 2, 3):
        cfg = I.small_configs()[idx]
        sc = O.Scenario(**I.scenario_kwargs(cfg))
        r = sc.simulate_stream(cfg["seed"], cfg["nu"], cfg["mask"])
        st = r["stream"]
        assert len(st) == r["stats"]["n_events"]                                   # one record per distinct executed event
        spec = st[st["loc2"] == 0xFFFFFFFF]
        assert len(spec) == r["richness"]
        ev = r["events"]                                                           # the speciation records ARE the species table
        assert np.array_equal(spec["loc"], ev["loc"]) and np.array_equal(spec["k"], ev["k"]) and np.array_equal(spec["f"], ev["f"])
        key = list(zip(st["k"].tolist(), st["f"].tolist(), st["loc"].tolist(), st["j"].tolist()))
        assert key == sorted(key) and len(set(key)) == len(key)                    # time order, no duplicates
        # closure under "the parent's lineage goes on": next event of loc2 after (k, f) is in the stream
        K = O.key_schedule(cfg["seed"])
        present = set(zip(st["loc"].tolist(), st["k"].tolist(), st["j"].tolist()))
        rng = np.random.default_rng(idx)
        disp = st[st["loc2"] != 0xFFFFFFFF]
        Cm, sh = O.turnover_scale(1.0, cfg["delta_t"])
        for rec in disp[rng.integers(0, len(disp), 300)]:
            if cfg["turnover"] is not None:
                continue                                                           # per-cell scales: covered by the uniform configs
            rc, k2, j2, T2, _ = O.next_event(K, int(rec["loc2"]), int(rec["k"]), int(rec["f"]), Cm, sh)
            assert rc == 0 and (int(rec["loc2"]), k2, j2) in present
        # every sampled individual's first event is there as well
        first = {}
        for rec in st:
            first.setdefault(int(rec["loc"]), (int(rec["k"]), int(rec["f"])))
        sampled = np.arange(sc.n_individuals) if cfg["mask"] is None else np.flatnonzero(cfg["mask"])
        assert all(int(l) in first for l in sampled[:200])
