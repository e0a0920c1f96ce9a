"""GPU parity of the Poisson / order-statistics event-time sampler against the oracle:
tables, the event-time search as a primitive, and the whole path with both simulate kernels -- bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
KERNELS = {"per_thread": 1, "tail": 0xFFFFFFFF}


@pytest.fixture(scope="module")
def ns():
    from paper_2108_05815_b200 import necsim
    necsim.lib()
    return necsim


@pytest.fixture(scope="module")
def I():
    from paper_2108_05815_b200 import inputs
    return inputs


def same(got, ref, tag=""):
    assert got["richness"] == ref["richness"], tag
    for f in ("loc", "k", "j", "f", "abundance", "time"):
        assert np.array_equal(got["events"][f], ref["events"][f]), (tag, f)
    assert np.array_equal(got["labels"], ref["labels"]), tag


def configs(I):
    rng = np.random.default_rng(5)
    out = [dict(I.scenario_kwargs(c), sampler=1) for c in I.small_configs()]
    masks = [c["mask"] for c in I.small_configs()]
    # large mu: more points per interval than the tail kernel's lanes (scalar continuation), with and without thinning
    out.append(dict(kind=I.NONSPATIAL, uniform_deme=400, uniform_turnover=12.0, delta_t=2.0, sampler=1)); masks.append(None)
    lam = rng.uniform(0.5, 6.0, 30 * 25)
    out.append(dict(kind=I.EXPLICIT_GAUSSIAN, width=30, height=25, uniform_deme=2, turnover=lam, sigma=1.2, delta_t=2.0, sampler=1)); masks.append(None)
    return out, masks


def test_tables_and_search_primitive(ns, O, I):
    rng = np.random.default_rng(1)
    kws, _ = configs(I)
    for kw in kws:
        g, o = ns.Scenario(**kw), O.Scenario(**kw)
        mu, pc, thin = g.debug_poisson_table()
        omu, opc = o.poisson_table()
        assert mu == omu and np.array_equal(pc, opc)
        hab_cells = np.arange(g.ncells) if kw.get("deme") is None else np.flatnonzero(np.asarray(kw["deme"]).ravel() > 0)
        assert all(int(thin[c]) == o.thin(int(c)) for c in rng.choice(hab_cells, min(len(hab_cells), 50)))   # habitat cells only
        n = 20_001
        cell = rng.integers(0, g.ncells, n).astype(np.uint32)
        if kw["kind"] >= I.EXPLICIT_MATRIX and kw.get("deme") is not None:
            hab = np.flatnonzero(np.asarray(kw["deme"]).ravel() > 0)
            cell = rng.choice(hab, n).astype(np.uint32)
        loc = rng.integers(0, 1 << 32, n, dtype=np.uint64).astype(np.uint32)
        k = rng.integers(0, 1 << 20, n).astype(np.uint32)
        f_last = rng.integers(-1, 1 << 48, n).astype(np.int64); f_last[::3] = -1
        gk, gj, gT, grc = g.debug_next_event_poisson(9, loc, cell, k, f_last)
        rk, rj, rT, rrc = o.batch_next_event_poisson(9, loc, cell, k, f_last)
        assert (grc == 0).all() and (rrc == 0).all()
        assert np.array_equal(gk, rk) and np.array_equal(gj, rj) and np.array_equal(gT, rT)
        g.close()


@pytest.mark.parametrize("kernel", sorted(KERNELS))
def test_whole_path(ns, O, I, kernel):
    kws, masks = configs(I)
    for idx, (kw, mask) in enumerate(zip(kws, masks)):
        nu = 5e-3
        o = O.Scenario(**kw)
        ref = o.simulate(3, nu, mask, dedup=True)
        sc = ns.Scenario(**kw)
        same(sc.simulate(3, nu, mask, tail_threshold=KERNELS[kernel]), ref, (idx, "dedup"))
        ref2 = o.simulate(3, nu, mask, dedup=False, per_lineage=True)
        got2 = sc.simulate(3, nu, mask, tail_threshold=KERNELS[kernel], dedup=False, per_lineage=True)
        same(got2, ref2, (idx, "nodedup"))
        for f in ("loc", "k", "j", "f"):
            assert np.array_equal(got2["per_lineage"][f], ref2["per_lineage"][f]), (idx, f)
        assert np.array_equal(got2["steps"], ref2["steps"])
        # launch-shape invariance (the reproducibility claim, L25)
        same(sc.simulate(3, nu, mask, block_threads=64, grid_blocks=3, dedup_log2_slots=6, epoch_events=200, dedup_probe=1), ref, (idx, "knobs"))
        sc.close()


def test_ewens_mean_gpu_poisson(ns):
    sc = ns.Scenario(ns.NONSPATIAL, uniform_deme=10_000, sampler=1)
    S = [sc.simulate(seed, 1e-3)["richness"] for seed in range(100)]
    assert abs(np.mean(S) - 69.6545) < 3 * 7.690 / 10.0, np.mean(S)
    sc.close()
