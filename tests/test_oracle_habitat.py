"""Pins of the oracle's temporally varying habitat ("temporally varying landscapes, which
enables simulating gradual habitat loss", reading R24): piecewise-constant deme maps ("eras"), the dispersal of an
event at interval k goes to habitat of the era in force at k.

  * an era with the same map as the present changes nothing, bit for bit;
  * no lineage is ever placed on a position that does not exist in the era of the event (checked on the full event stream);
  * species-abundance distribution and richness against the Classical algorithm WITH its global clock and the same switch of maps
    (tests/classical.py::simulate_classical_timed) -- and far from the static results of either map alone, so that an era that is
    ignored, or applied at the wrong time, fails;
  * the arguments are validated (habitat may only be lost towards the present).
"""
import numpy as np
import pytest
from scipy import stats

from classical import simulate_classical_timed, sad_of
from test_oracle_model import _compare_sad

EXPLICIT_GAUSSIAN = 3


def landscape():
    W = H = 8
    rng = np.random.default_rng(21)
    present = np.zeros(W * H, np.uint32)
    present[rng.choice(W * H, 20, replace=False)] = 2          # what is left today: 20 cells of 2
    past = np.full(W * H, 3, np.uint32)                        # before the loss: habitat everywhere, demes of 3
    return W, H, present, past


def test_same_map_in_the_past_changes_nothing(O):
    W, H, present, _ = landscape()
    a = O.Scenario(EXPLICIT_GAUSSIAN, W, H, deme=present, sigma=0.5, delta_t=1.0)
    b = O.Scenario(EXPLICIT_GAUSSIAN, W, H, deme=present, sigma=0.5, delta_t=1.0, past_deme=[present, present], past_start_k=[3, 11])
    assert a.n_individuals == b.n_individuals == int(present.sum())
    for seed in range(20):
        ra, rb = a.simulate(seed, 0.05), b.simulate(seed, 0.05)
        assert ra["richness"] == rb["richness"] and (ra["events"] == rb["events"]).all() and (ra["labels"] == rb["labels"]).all()


def test_never_outside_the_habitat_of_the_era(O):
    W, H, present, past = landscape()
    mid = np.maximum(present, (np.arange(W * H) % 3 == 0).astype(np.uint32) * 3)      # a middle era: nested between the two
    starts = [4, 9]
    sc = O.Scenario(EXPLICIT_GAUSSIAN, W, H, deme=present, sigma=0.7, delta_t=1.0, past_deme=[mid, past], past_start_k=starts)
    maps = [present, mid, past]
    prefix = np.concatenate([[0], np.cumsum(past)])                                  # locations are canonical on the oldest map
    seen_eras = set()
    for seed in range(30):
        r = sc.simulate_stream(seed, 0.02)
        st = r["stream"]
        cell = np.searchsorted(prefix, st["loc"], side="right") - 1
        idx = st["loc"] - prefix[cell]
        era = np.searchsorted(np.array([0] + starts), st["k"], side="right") - 1
        seen_eras |= set(era.tolist())
        for e in range(3):
            m = era == e
            assert (idx[m] < maps[e][cell[m]]).all()                                 # the individual that has the event exists in its era
            d = m & (st["loc2"] != 0xFFFFFFFF)
            c2 = np.searchsorted(prefix, st["loc2"][d], side="right") - 1
            assert (st["loc2"][d] - prefix[c2] < maps[e][c2]).all()                  # and so does the parent it came from
    assert seen_eras == {0, 1, 2}


def test_sad_vs_classical_with_habitat_loss(O):
    W, H, present, past = landscape()
    sigma, nu, dt, k_c, n = 0.7, 0.06, 1.0, 2, 3000
    sc = O.Scenario(EXPLICIT_GAUSSIAN, W, H, deme=present, sigma=sigma, delta_t=dt, past_deme=[past], past_start_k=[k_c])
    o_sads, o_S = [], []
    for seed in range(n):
        r = sc.simulate(seed, nu); o_sads.append(np.bincount(r["events"]["abundance"])); o_S.append(r["richness"])

    def disperse_at(g, l, t):
        deme = past if t >= k_c * dt else present
        cell, _ = l
        x0, y0 = cell % W, cell // W
        while True:
            dx = int(np.rint(g.normal(0.0, sigma))); dy = int(np.rint(g.normal(0.0, sigma)))
            c2 = ((y0 + dy) % H) * W + (x0 + dx) % W
            if deme[c2] > 0:
                return (c2, int(g.integers(deme[c2])))
    starts = [(c, i) for c in range(W * H) for i in range(present[c])]
    rng = np.random.default_rng(8)
    c_sads, c_S = [], []
    for _ in range(n):
        lab = simulate_classical_timed(rng, starts, nu, disperse_at)
        c_sads.append(sad_of(lab)); c_S.append(len(set(lab)))
    assert _compare_sad(o_sads, c_sads, 12) > 1e-3
    assert stats.ks_2samp(o_S, c_S).pvalue > 1e-3
    se = np.sqrt(np.var(o_S) / n + np.var(c_S) / n)
    assert abs(np.mean(o_S) - np.mean(c_S)) < 4 * se
    # the switch matters: the static present-day landscape (no era) and a switch at the wrong time are many standard errors away
    for wrong in (dict(), dict(past_deme=[past], past_start_k=[12])):
        w = O.Scenario(EXPLICIT_GAUSSIAN, W, H, deme=present, sigma=sigma, delta_t=dt, **wrong)
        S = [w.simulate(seed, nu)["richness"] for seed in range(n)]
        assert abs(np.mean(S) - np.mean(c_S)) > 8 * se, (wrong.get("past_start_k"), np.mean(S), np.mean(c_S))


def test_eras_are_validated(O):
    W, H, present, past = landscape()
    bad = past.copy(); bad[np.flatnonzero(present)[0]] = 1                            # less habitat in the past than today
    for kw in (dict(past_deme=[bad], past_start_k=[3]), dict(past_deme=[past], past_start_k=[0]),
               dict(past_deme=[past, past], past_start_k=[5, 5])):
        with pytest.raises(ValueError):
            O.Scenario(EXPLICIT_GAUSSIAN, W, H, deme=present, sigma=0.5, delta_t=1.0, **kw)
    with pytest.raises(ValueError):
        O.Scenario(0, 1, 1, uniform_deme=10, past_deme=[np.array([10], np.uint32)], past_start_k=[2])      # gaussian kind only
