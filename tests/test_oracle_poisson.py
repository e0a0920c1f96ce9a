"""Pins of the oracle's Poisson / order-statistics event-time sampler (PAPER.md 5.2.3 L733-741, C.5
L1940-1954). None of these re-types the oracle's arithmetic: they check what the mathematics fixes -- the Poisson law of
the counts, exponential gaps (L1206), the alignment property (L715, L729), exact thinning rates, and the Ewens mean."""
import numpy as np
import pytest
from scipy import stats


def test_cdf_table_against_scipy(O):
    for mu in (0.5, 2.0, 7.3, 40.0):
        sc = O.Scenario(O.NONSPATIAL, uniform_deme=10, uniform_turnover=mu / 2.0, delta_t=2.0, sampler=1)
        m, PC = sc.poisson_table()
        assert m == mu
        ref = stats.poisson.cdf(np.arange(256), mu)
        got = PC.astype(np.float64) / 2.0**64
        assert np.all(np.abs(got - ref) < 1e-13)
        assert np.all(np.diff(PC.astype(np.float64)) >= 0)


def _walk_stream(sc, seed, loc, cell, n_events):
    """Consecutive events of ONE location's stream (no dispersal): (k, j, T) sequence via repeated next_event."""
    k, f, out = 0, -1, []
    for _ in range(n_events):
        ko, jo, To, rc = sc.batch_next_event_poisson(seed, np.array([loc], np.uint32), cell, k, f)
        assert rc[0] == 0
        k, f = int(ko[0]), int(To[0])
        out.append((k, int(jo[0]), f))
    return out


def test_gaps_are_exponential_and_counts_poisson(O):
    lam, dt = 0.8, 2.0
    sc = O.Scenario(O.NONSPATIAL, uniform_deme=50, uniform_turnover=lam, delta_t=dt, sampler=1)
    ev = _walk_stream(sc, 11, 7, 0, 6000)
    t = np.array([(k + f / 2.0**48) * dt for k, _, f in ev])
    assert np.all(np.diff(t) > 0)
    assert stats.kstest(np.diff(t), "expon", args=(0, 1.0 / lam)).pvalue > 1e-3            # turnover test, L1206
    ks = np.array([k for k, _, _ in ev])
    counts = np.bincount(ks)[: ks.max()]                                                      # complete intervals only
    mu = lam * dt
    exp = stats.poisson.pmf(np.arange(8), mu) * len(counts)
    obs = np.array([np.sum(counts == n) for n in range(8)])
    assert stats.chisquare(obs[:6], exp[:6] * obs[:6].sum() / exp[:6].sum()).pvalue > 1e-3
    within = np.array([f / 2.0**48 for _, _, f in ev])
    assert stats.kstest(within, "uniform").pvalue > 1e-3                                      # order statistics: uniform offsets, L737


def test_thinning_gives_each_cell_its_own_rate(O):
    """Per-cell turnover: the stream of a cell with lambda < lambda_max is the lambda_max stream thinned by lambda/lambda_max."""
    lam = np.array([0.5, 1.0, 2.0, 1.5])
    sc = O.Scenario(O.EXPLICIT_GAUSSIAN, width=2, height=2, uniform_deme=1, turnover=lam, sigma=0.05, delta_t=1.0, sampler=1)
    assert sc.thin(2) == 0xFFFFFFFF and sc.thin(0) == 2**30 and sc.thin(3) == 3 * 2**30
    for cell in range(4):
        ev = _walk_stream(sc, 5, cell, cell, 3000)                       # deme 1: loc == cell
        t = np.array([(k + f / 2.0**48) * 1.0 for k, _, f in ev])
        assert stats.kstest(np.diff(t), "expon", args=(0, 1.0 / lam[cell])).pvalue > 1e-3


def test_alignment_two_arrivals_find_the_same_next_event(O):
    """A lineage arriving between two points of a stream finds the later point, whatever its arrival time (L715, L729)."""
    sc = O.Scenario(O.NONSPATIAL, uniform_deme=50, uniform_turnover=1.3, delta_t=2.0, sampler=1)
    rng = np.random.default_rng(3)
    ev = _walk_stream(sc, 21, 3, 0, 400)
    for (k0, _, f0), (k1, j1, f1) in zip(ev[:-1], ev[1:]):
        if k0 != k1:
            continue
        for f in rng.integers(f0, f1, 3):                              # f0 <= f < f1: strictly before the next point
            ko, jo, To, rc = sc.batch_next_event_poisson(21, np.array([3], np.uint32), 0, k0, int(f))
            assert (int(ko[0]), int(jo[0]), int(To[0])) == (k1, j1, f1)
        ko, jo, To, rc = sc.batch_next_event_poisson(21, np.array([3], np.uint32), 0, k1, f1)   # strictness: not itself
        assert (int(ko[0]), int(To[0])) != (k1, f1)


def test_ewens_mean_and_tiny_closed_forms(O):
    sc = O.Scenario(O.NONSPATIAL, uniform_deme=10_000, sampler=1)
    S = [sc.simulate(seed, 1e-3)["richness"] for seed in range(100)]
    assert abs(np.mean(S) - 69.6545) < 3 * 7.690 / 10.0                 # Eq. B.1 with theta = J nu / (1 - nu)
    sc2 = O.Scenario(O.NONSPATIAL, uniform_deme=3, sampler=1)
    S2 = [sc2.simulate(seed, 0.5)["richness"] for seed in range(20000)]
    assert abs(np.mean(S2) - 2.35) < 0.02                               # sum_i theta / (theta + i), J = 3, nu = 0.5


def test_dedup_on_off_and_sampler_changes_realisation_not_law(O, ):
    from paper_2108_05815_b200 import inputs as I
    cfg = I.small_configs()[3]
    kw = dict(I.scenario_kwargs(cfg), sampler=1)
    sc = O.Scenario(**kw)
    a = sc.simulate(cfg["seed"], 5e-3, cfg["mask"], dedup=True)
    b = sc.simulate(cfg["seed"], 5e-3, cfg["mask"], dedup=False)
    c = sc.simulate(cfg["seed"], 5e-3, cfg["mask"], dedup=True, epoch_events=500)
    for r in (b, c):
        assert r["richness"] == a["richness"] and np.array_equal(r["labels"], a["labels"])
        assert all(np.array_equal(r["events"][f], a["events"][f]) for f in ("loc", "k", "j", "f", "abundance", "time"))
    e = O.Scenario(**dict(kw, sampler=0)).simulate(cfg["seed"], 5e-3, cfg["mask"], dedup=True)
    assert not np.array_equal(e["events"]["f"][: min(5, e["richness"])], a["events"]["f"][: min(5, a["richness"])])
