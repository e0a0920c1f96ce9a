"""Pin of the output ORDER and the label ranks (reading R22; the stream is ordered by
event time; L962-967: duplicates of an event are merged).

The expected table is built here, in Python, from the per-lineage terminal records of a dedup-off run: every lineage then
walks its own path to its own speciation event, and nothing of the oracle's comparator (`cmp_event`), its unique pass or
its label search is involved. Sorting those records by (k, f, loc, j) with Python tuples must reproduce `events`,
`labels` and `abundance` of the dedup-on run. A comparator that orders by another field first, or descending, fails here.
"""
import numpy as np

from paper_2108_05815_b200 import inputs as I


def expected_table(per_lineage):
    keys = [(int(r["k"]), int(r["f"]), int(r["loc"]), int(r["j"])) for r in per_lineage]
    uniq = sorted(set(keys))                                   # Python tuple order = (k, f, loc, j) ascending
    rank = {key: i for i, key in enumerate(uniq)}
    labels = np.array([rank[key] for key in keys], dtype=np.uint32)
    abundance = np.bincount(labels, minlength=len(uniq)).astype(np.uint32)
    return uniq, labels, abundance


def check(O, cfg):
    sc = O.Scenario(**I.scenario_kwargs(cfg))
    nd = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=False, per_lineage=True)
    uniq, labels, abundance = expected_table(nd["per_lineage"])
    for mode in (dict(dedup=True), dict(dedup=True, epoch_events=500), dict(dedup=False)):
        r = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], **mode)
        ev = r["events"]
        assert r["richness"] == len(uniq)
        assert [(int(e["k"]), int(e["f"]), int(e["loc"]), int(e["j"])) for e in ev] == uniq
        assert np.array_equal(r["labels"], labels)
        assert np.array_equal(ev["abundance"], abundance)
        # times follow the order (ties in (k, f) are possible in principle, so non-strict)
        assert np.all(np.diff(ev["time"]) >= 0)
    return uniq


def test_order_and_ranks_small_configs(O):
    for cfg in I.small_configs():
        uniq = check(O, cfg)
        assert len(uniq) >= 3


def test_order_distinguishes_the_key_fields(O):
    """A workload with many species, so that the order by (k, f) differs from the order by loc, by j and by f alone."""
    cfg = I.c1_nonspatial(J=400, nu=0.05, seed=3)
    uniq = check(O, cfg)
    assert len(uniq) > 40
    ks = [u[0] for u in uniq]; fs = [u[1] for u in uniq]; locs = [u[2] for u in uniq]
    assert len(set(ks)) < len(ks), "several events must share an interval k for f to matter"
    assert sorted(fs) != fs, "ordering by f alone must differ from (k, f)"
    assert sorted(locs) != locs and sorted(locs, reverse=True) != locs, "ordering by loc must differ"
    cfg = I.c4_gaussian(side=31, sigma=1.5, nu=0.02, seed=5)
    check(O, cfg)
