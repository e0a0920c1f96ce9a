"""GPU parity on the rarer code paths of both simulate kernels (bit-exact against the oracle):
large mu (more than 16 points per interval: the tail kernel's scalar continuation), demes >= 255 (deme32 path),
matrix dispersal with per-cell turnover and non-habitat cells, wide sigma (crowded guide buckets -> exact forward
scan), non-power-of-two and non-square tori, migration 0 and 1, a step cap together with dedup."""
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


def same(got, ref):
    assert got["richness"] == ref["richness"]
    for f in ("loc", "k", "j", "f", "abundance", "time"):
        assert np.array_equal(got["events"][f], ref["events"][f]), f
    assert np.array_equal(got["labels"], ref["labels"])


def scenarios(I):
    rng = np.random.default_rng(99)
    out = []
    # (a) mu = 40: ~40 points per interval
    out.append(("mu40-nonspatial", dict(kind=I.NONSPATIAL, uniform_deme=500, uniform_turnover=20.0, delta_t=2.0), 0.01, None))
    out.append(("mu40-gauss", dict(kind=I.EXPLICIT_GAUSSIAN, width=40, height=33, uniform_deme=2, uniform_turnover=8.0, delta_t=5.0, sigma=1.5), 0.01, None))
    # (b) demes up to 1000 (deme32 path), some non-habitat, non-pow2 / non-square torus
    deme = rng.integers(0, 4, 47 * 31).astype(np.uint32)
    deme[rng.integers(0, len(deme), 25)] = rng.integers(255, 1000, 25)
    out.append(("deme32-gauss", dict(kind=I.EXPLICIT_GAUSSIAN, width=47, height=31, deme=deme, sigma=2.0, delta_t=2.0), 0.005, None))
    # (c) matrix + per-cell turnover + non-habitat cells + one big deme
    n = 9 * 7
    d2 = rng.integers(0, 6, n).astype(np.uint32); d2[3] = 300; d2[d2.argmax()] = 300
    w = rng.random((n, n)) * (d2[None, :] > 0)
    w[:, 3] += 0.5
    turn = 0.3 + 2.0 * rng.random(n)
    out.append(("matrix-percell", dict(kind=I.EXPLICIT_MATRIX, width=9, height=7, deme=d2, matrix=w, turnover=turn, delta_t=1.0), 0.01, None))
    # (d) wide sigma: 2R = 240 thresholds over 2048 guide buckets
    hab = (rng.random(150 * 130) < 0.8).astype(np.uint32) * 3
    out.append(("sigma12", dict(kind=I.EXPLICIT_GAUSSIAN, width=150, height=130, deme=hab, sigma=12.0, turnover=0.5 + rng.random(150 * 130), delta_t=2.0), 0.004,
                (rng.random(int(hab.sum())) < 0.2).astype(np.uint8)))
    # (e) implicit: everyone migrates at once / nobody ever migrates (then nu applies nowhere: needs the step cap)
    out.append(("implicit-m1", dict(kind=I.SPATIALLY_IMPLICIT, local_size=700, meta_size=5000, migration=1.0), 0.02, None))
    return out


@pytest.mark.parametrize("kernel", sorted(KERNELS))
def test_rare_paths(ns, O, I, kernel):
    for name, kw, nu, mask in scenarios(I):
        ref = O.Scenario(**kw).simulate(5, nu, mask, dedup=True)
        sc = ns.Scenario(**kw)
        got = sc.simulate(5, nu, mask, tail_threshold=KERNELS[kernel])
        same(got, ref)
        got2 = sc.simulate(5, nu, mask, tail_threshold=KERNELS[kernel], dedup=False, per_lineage=True)
        ref2 = O.Scenario(**kw).simulate(5, nu, mask, dedup=False, per_lineage=True)
        same(got2, ref2)
        for f in ("loc", "k", "j", "f"):
            assert np.array_equal(got2["per_lineage"][f], ref2["per_lineage"][f]), (name, f)
        assert np.array_equal(got2["steps"], ref2["steps"]), name
        sc.close()


def test_bigdeme_shape_next4(ns, O, I):
    """few cells with enormous demes (every deme >= 255: the deme32 gather on every dispersal)."""
    cfg = I.c6_bigdeme(width=24, height=21, deme_mean=2000, sigma=1.0, nu=5e-3, sample=0.02, seed=3)
    kw = I.scenario_kwargs(cfg)
    ref = O.Scenario(**kw).simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True)
    sc = ns.Scenario(**kw)
    for knobs in (dict(), dict(tail_threshold=1), dict(tail_threshold=0xFFFFFFFF)):
        same(sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], **knobs), ref)
    sc.close()
    kw1 = dict(kw, sampler=1)
    same(ns.Scenario(**kw1).simulate(cfg["seed"], cfg["nu"], cfg["mask"]), O.Scenario(**kw1).simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True))


@pytest.mark.parametrize("kernel", sorted(KERNELS))
def test_step_cap_with_dedup_and_no_migration(ns, O, I, kernel):
    kw = dict(kind=I.SPATIALLY_IMPLICIT, local_size=300, meta_size=1000, migration=0.0)
    ref = O.Scenario(**kw).simulate(9, 0.5, None, dedup=True, max_steps=50)
    sc = ns.Scenario(**kw)
    got = sc.simulate(9, 0.5, None, max_steps=50, tail_threshold=KERNELS[kernel], dedup_probe=1)
    # nobody can speciate in the local community (nu = 0 there, L1830): everything unfinished or culled into an unfinished lineage
    assert got["richness"] == ref["richness"] == 0
    assert (got["labels"] == 0xFFFFFFFF).all() and (ref["labels"] == 0xFFFFFFFF).all()
    sc.close()
