"""GPU parity, primitive by primitive, through the necsim_debug_* exports of the C-ABI (bit-exact vs the oracle).
Localises a mismatch of the whole path to hash / -ln / event-time search / dispersal / tables."""
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


def test_draws_bit_exact(ns, O):
    rng = np.random.default_rng(1)
    n = 100_003                                    # several blocks and a ragged tail
    loc = rng.integers(0, 1 << 32, n, dtype=np.uint64).astype(np.uint32)
    k = rng.integers(0, 1 << 32, n, dtype=np.uint64).astype(np.uint32)
    j = rng.integers(1, 200, n).astype(np.uint32)
    r = rng.integers(0, 50, n).astype(np.uint32)
    for seed in (0, 42, 2**64 - 1):
        for lane in ("state", "time", "spec", "disp", "index", "migr"):
            got = ns.debug_draw(seed, lane, loc, k, j, r)
            ref = O.batch_draw(seed, lane, loc, k, j, r)
            assert np.array_equal(got, ref), (seed, lane)


def test_neglog_bit_exact(ns, O):
    rng = np.random.default_rng(2)
    x = rng.integers(0, 1 << 64, 200_001, dtype=np.uint64)
    edge = np.array([0, 1, 2, 3, 2**64 - 1, 2**63, 2**63 - 1, 2**63 + 1, 2**32, 2**32 - 1, 2**14, 2**14 - 1], dtype=np.uint64)
    small = (x >> rng.integers(0, 64, len(x)).astype(np.uint64))     # exercise every leading-zero count
    x = np.concatenate([edge, x, small])
    assert np.array_equal(ns.debug_neglog(x), O.batch_neglog(x))


def test_next_event_bit_exact(ns, O):
    rng = np.random.default_rng(3)
    n = 50_001
    loc = rng.integers(0, 1 << 32, n, dtype=np.uint64).astype(np.uint32)
    k = rng.integers(0, 1 << 20, n).astype(np.uint32)
    f_last = rng.integers(-1, 1 << 48, n).astype(np.int64)
    f_last[::3] = -1
    lam = rng.uniform(0.2, 3.0, n)
    cs = [O.turnover_scale(l, 2.0) for l in lam]
    Cm = np.array([c[0] for c in cs], np.uint32); sh = np.array([c[1] for c in cs], np.uint32)
    gk, gj, gT, grc = ns.debug_next_event(7, loc, k, f_last, Cm, sh)
    rk, rj, rT, rrc = O.batch_next_event(7, loc, k, f_last, Cm, sh)
    assert np.array_equal(grc, rrc) and (grc == 0).all()
    assert np.array_equal(gk, rk) and np.array_equal(gj, rj) and np.array_equal(gT, rT)


def test_tables_and_dispersal_bit_exact(ns, O, I):
    rng = np.random.default_rng(4)
    for cfg in I.small_configs():
        kw = I.scenario_kwargs(cfg)
        g, o = ns.Scenario(**kw), O.Scenario(**kw)
        assert g.n_individuals == o.n_individuals
        t = g.debug_tables()
        if cfg["kind"] == I.EXPLICIT_MATRIX:
            th, al = o.alias_tables()
            assert np.array_equal(t["thresh"], th) and np.array_equal(t["alias"], al)
        if cfg["kind"] == I.EXPLICIT_GAUSSIAN:
            R, TG = O.gauss_table(cfg["sigma"])
            assert t["R"] == R and np.array_equal(t["gauss"], TG)
        if cfg["turnover"] is not None:
            deme = np.asarray(cfg["deme"]).ravel()
            for c in rng.integers(0, len(deme), 200):
                if deme[c]:
                    assert (t["Cm"][c], t["sh"][c]) == O.turnover_scale(cfg["turnover"].ravel()[c], cfg["delta_t"])
        n = 20_001
        n_loc = g.n_individuals if cfg["kind"] != I.SPATIALLY_IMPLICIT else cfg["local_size"] + cfg["meta_size"]
        loc = rng.integers(0, n_loc, n).astype(np.uint32)
        k = rng.integers(0, 1000, n).astype(np.uint32); j = rng.integers(1, 9, n).astype(np.uint32)
        assert np.array_equal(g.debug_disperse(cfg["seed"], loc, k, j), O.batch_disperse(o, cfg["seed"], loc, k, j)), cfg["name"]
        g.close()


def test_fast_round_filter_error_bound(ns, O):
    """The tail kernel's fast round compares binary32 offsets (top 32 bits of a draw, lg2.approx) and only trusts a comparison
    further than `margin` from equality. Pin of that filter: over the draws it accepts (2^20 <= hi < 2^32 - 2^8)
    the binary32 offset is within margin / 8 of the exact Q16.48 offset of DESIGN.md 2.4 (taken from the ORACLE), for turnover
    scales over the whole admissible range of mu; partial sums of up to five terms then stay within margin / 1.6."""
    rng = np.random.default_rng(11)
    n = 2_000_003
    x = rng.integers(0, 1 << 64, n, dtype=np.uint64)
    x[: n // 4] |= np.uint64(0xFFF0_0000_0000_0000)                      # many draws near U = 1 (tiny offsets)
    q = n // 4
    x[q: 2 * q] >>= rng.integers(0, 12, q).astype(np.uint64)             # small U (large offsets), down to hi = 2^20
    hi = x >> np.uint64(32)
    ok = (hi >= (1 << 20)) & (hi < (1 << 32) - (1 << 8))
    x = x[ok]
    E = O.batch_neglog(x)
    for lam_dt in (1.0 / 200, 0.1, 0.5, 1.0, 2.0, 3.0, 17.0, 64.0):
        Cm, sh = O.turnover_scale(lam_dt, 1.0)
        ap, ex, margin = ns.debug_approx_time(x, Cm, sh)
        ref = np.array([O.scale(int(e), Cm, sh) for e in E[:2000]], dtype=np.uint64)
        assert np.array_equal(ex[:2000], ref)                            # the exact side of the export is the oracle's arithmetic
        t = ex.astype(np.float64) * 2.0 ** -48
        rel = t < 2.0                                                    # offsets that can take part in a decision (sums near <= 1)
        err = np.abs(ap.astype(np.float64) - t)[rel]
        assert err.size > 1000 and err.max() <= margin / 8.0, (lam_dt, err.max(), margin)
    # zero increments cannot hide behind an accepted draw: hi < 2^32 - 2^8 means an exact offset > 0
    Cm, sh = O.turnover_scale(64.0, 1.0)
    _, ex, _ = ns.debug_approx_time(x, Cm, sh)
    assert (ex > 0).all()
