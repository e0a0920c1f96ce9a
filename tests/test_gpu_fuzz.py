"""Randomised GPU-vs-oracle parity: many seeds and many small random scenarios (all four kinds, random sizes, demes,
turnover, sigma, masks, launch knobs), plus the Ewens pin (PAPER.md Eq. B.1) applied to the GPU path itself."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ns():
    from paper_2108_05815_b200 import necsim
    necsim.lib()
    return necsim


@pytest.fixture(scope="module")
def I():
    from paper_2108_05815_b200 import inputs
    return inputs


def same(got, ref, tag):
    assert got["richness"] == ref["richness"], tag
    for f in ("loc", "k", "j", "f", "abundance", "time"):
        assert np.array_equal(got["events"][f], ref["events"][f]), (tag, f)
    assert np.array_equal(got["labels"], ref["labels"]), tag


def random_scenario(I, rng):
    kind = int(rng.integers(0, 4))
    dt = float(rng.choice([0.5, 1.0, 2.0, 3.0]))
    if kind == I.NONSPATIAL:
        return dict(kind=kind, uniform_deme=int(rng.integers(1, 400)), uniform_turnover=float(rng.uniform(0.3, 3.0)), delta_t=dt)
    if kind == I.SPATIALLY_IMPLICIT:
        return dict(kind=kind, local_size=int(rng.integers(1, 300)), meta_size=int(rng.integers(1, 5000)),
                    migration=float(rng.choice([0.01, 0.1, 0.5, 1.0])), uniform_turnover=float(rng.uniform(0.3, 3.0)), delta_t=dt)
    w, h = int(rng.integers(1, 14)), int(rng.integers(1, 14))
    n = w * h
    deme = rng.integers(0, 5, n).astype(np.uint32)
    deme[int(rng.integers(0, n))] = int(rng.integers(1, 6))          # at least one habitat cell
    turnover = None if rng.random() < 0.5 else rng.uniform(0.3, 3.0, n)
    if kind == I.EXPLICIT_MATRIX:
        m = rng.random((n, n)) * (rng.random((n, n)) < 0.5) * (deme[None, :] > 0)
        m[:, int(np.flatnonzero(deme)[0])] += 0.1                    # every row has mass on a habitat column
        return dict(kind=kind, width=w, height=h, deme=deme, matrix=m, turnover=turnover, delta_t=dt)
    w, h = int(rng.integers(12, 40)), int(rng.integers(12, 40))
    n = w * h
    sigma = float(rng.uniform(0.3, 1.1))                             # R = ceil(10 sigma) < min(w, h)
    deme = (rng.random(n) < rng.uniform(0.3, 1.0)).astype(np.uint32) * rng.integers(1, 4, n).astype(np.uint32)
    deme[int(rng.integers(0, n))] = 1
    turnover = None if rng.random() < 0.5 else rng.uniform(0.3, 3.0, n)
    return dict(kind=kind, width=w, height=h, deme=deme, sigma=sigma, turnover=turnover, delta_t=dt)


def test_random_scenarios(ns, O, I):
    rng = np.random.default_rng(2024)
    import os
    for case in range(int(os.environ.get("NECSIM_FUZZ_CASES", "60"))):
        kw = random_scenario(I, rng)
        o = O.Scenario(**kw)
        n_ind = o.n_individuals
        mask = None
        if rng.random() < 0.5 and n_ind > 1:
            mask = (rng.random(n_ind) < rng.uniform(0.2, 0.9)).astype(np.uint8)
            mask[int(rng.integers(0, n_ind))] = 1
        nu = float(rng.choice([1.0, 0.3, 0.05, 0.01]))
        seed = int(rng.integers(0, 2**63))
        kw["sampler"] = int(rng.integers(0, 2))                       # exponential or Poisson event-time sampler
        record = bool(rng.integers(0, 2))                             # with or without the full event stream
        knobs = dict(tail_threshold=int(rng.choice([1, 0xFFFFFFFF, 0])), dedup_probe=int(rng.integers(0, 8)),
                     dedup_log2_slots=int(rng.choice([4, 8, 16, 0])), block_threads=int(rng.choice([32, 128, 256])),
                     epoch_events=int(rng.choice([0, 1, 50, 5000])))
        o = O.Scenario(**kw)
        ref = o.simulate_stream(seed, nu, mask) if record else o.simulate(seed, nu, mask, dedup=True)
        sc = ns.Scenario(**kw)
        if record:
            knobs.update(record_events=True, event_ring_capacity=int(rng.choice([1 << 16, 1 << 20])), event_stream_capacity=1 << 21)
        got = sc.simulate(seed, nu, mask, **knobs)
        same(got, ref, (case, kw["kind"], knobs))
        if record:
            assert len(got["stream"]) == len(ref["stream"]), (case, knobs)
            for f in ("loc", "k", "j", "f", "loc2"):
                assert np.array_equal(got["stream"][f], ref["stream"][f]), (case, knobs, f)
        sc.close()


def test_many_seeds_small_configs(ns, O, I):
    for cfg in I.small_configs()[:4]:
        kw = I.scenario_kwargs(cfg)
        o, sc = O.Scenario(**kw), ns.Scenario(**kw)
        for seed in range(100, 106):
            nu = max(cfg["nu"], 2e-3)
            same(sc.simulate(seed, nu, cfg["mask"]), o.simulate(seed, nu, cfg["mask"], dedup=True), (cfg["name"], seed))
        sc.close()


def test_ewens_mean_on_the_gpu_path(ns):
    """C1 (J = 1e4, nu = 1e-3): E[S] = theta (psi(theta + J) - psi(theta)) = 69.6545, sd 7.69: the GPU mean over
    100 seeds must lie within 3 standard errors."""
    sc = ns.Scenario(ns.NONSPATIAL, uniform_deme=10_000)
    S = [sc.simulate(seed, 1e-3)["richness"] for seed in range(100)]
    assert abs(np.mean(S) - 69.6545) < 3 * 7.690 / 10.0, np.mean(S)
    sc.close()
