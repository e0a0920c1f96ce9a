"""GPU parity of the temporally varying habitat against the oracle's era mode
(pinned in tests/test_oracle_habitat.py): both kernels, both event-time samplers, dedup on / off, epochs, the event stream."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
GAUSS = 3


def scenarios():
    rng = np.random.default_rng(31)
    out = []
    # (a) deme 2 today on a third of the cells, 3 everywhere in the past; two switches
    W, H = 37, 29
    now = np.zeros(W * H, np.uint32); now[rng.choice(W * H, W * H // 3, replace=False)] = 2
    mid = np.maximum(now, (rng.random(W * H) < 0.5).astype(np.uint32) * 2)
    old = np.full(W * H, 3, np.uint32)
    out.append(dict(kind=GAUSS, width=W, height=H, deme=now, sigma=1.6, delta_t=2.0, past_deme=np.stack([mid, old]), past_start_k=[3, 9]))
    # (b) per-cell turnover, demes beyond 255 (deme32 tables per era), one switch
    W, H = 24, 24
    now = (rng.random(W * H) < 0.4).astype(np.uint32) * rng.integers(1, 400, W * H).astype(np.uint32)
    now[5] = 300
    old = np.maximum(now, rng.integers(0, 500, W * H).astype(np.uint32))
    out.append(dict(kind=GAUSS, width=W, height=H, deme=now, turnover=0.5 + rng.random(W * H), sigma=1.1, delta_t=1.5,
                    past_deme=old[None, :], past_start_k=[4]))
    return out


@pytest.mark.parametrize("idx", [0, 1])
@pytest.mark.parametrize("sampler", [0, 1])
def test_eras_match_oracle(O, idx, sampler):
    from paper_2108_05815_b200 import necsim as ns
    kw = dict(scenarios()[idx], sampler=sampler)
    nu, seed = 3e-3, 77 + idx
    osc, sc = O.Scenario(**kw), ns.Scenario(**kw)
    assert sc.n_individuals == osc.n_individuals == int(np.asarray(kw["deme"]).sum())
    rng = np.random.default_rng(idx)
    mask = (rng.random(sc.n_individuals) < 0.6).astype(np.uint8)
    ref = osc.simulate(seed, nu, mask, dedup=True)
    for p in (dict(), dict(tail_threshold=1), dict(tail_threshold=10**9), dict(epoch_events=3000), dict(epoch_events=700, tail_threshold=1),
              dict(dedup=False, tail_threshold=1), dict(dedup=False, tail_threshold=10**9), dict(grid_blocks=3, block_threads=64, dedup_log2_slots=8)):
        got = sc.simulate(seed, nu, mask, **p)
        assert got["richness"] == ref["richness"], p
        for f in ("loc", "k", "j", "f", "abundance", "time"):
            assert np.array_equal(got["events"][f], ref["events"][f]), (p, f)
        assert np.array_equal(got["labels"], ref["labels"]), p
    # per-lineage terminal records with dedup off, and the full event stream
    nd_ref = osc.simulate(seed, nu, mask, dedup=False, per_lineage=True)
    for tt in (1, 10**9):
        nd = sc.simulate(seed, nu, mask, per_lineage=True, dedup=False, tail_threshold=tt)
        for f in ("loc", "k", "j", "f"):
            assert np.array_equal(nd["per_lineage"][f], nd_ref["per_lineage"][f]), (tt, f)
        assert np.array_equal(nd["steps"], nd_ref["steps"])
    st_ref = osc.simulate_stream(seed, nu, mask)["stream"]
    for tt in (1, 10**9):
        st = sc.simulate(seed, nu, mask, record_events=True, event_ring_capacity=1 << 18, event_stream_capacity=1 << 23, tail_threshold=tt)["stream"]
        assert len(st) == len(st_ref)
        for f in ("loc", "k", "j", "f", "loc2"):
            assert np.array_equal(st[f], st_ref[f]), (tt, f)
    sc.close()


def test_era_arguments_are_validated():
    from paper_2108_05815_b200 import necsim as ns
    base = scenarios()[0]
    bad = dict(base); bad["past_deme"] = np.stack([base["past_deme"][1], base["past_deme"][0]])     # not nested
    with pytest.raises(ns.NecsimError):
        ns.Scenario(**bad)
    bad = dict(base); bad["past_start_k"] = [3, 3]
    with pytest.raises(ns.NecsimError):
        ns.Scenario(**bad)
    with pytest.raises(ns.NecsimError):
        ns.Scenario(kind=0, uniform_deme=10, past_deme=np.array([[10]], np.uint32), past_start_k=[2])
