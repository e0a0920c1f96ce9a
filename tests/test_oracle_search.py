"""P3/P4 -- event-time search (PAPER.md 5.2.2-5.2.3 L709-741) and speciation test
(Fig. 5.1): exact alignment properties by brute force, and the paper's own event statistics
(L1200-1208): turnover times ~ Exp(lambda), points per interval ~ Poisson(lambda*dt), speciation times
~ Exp(lambda*nu) with dispersal disabled."""
import numpy as np
from scipy import stats

TWO48 = 1 << 48


def enumerate_interval(O, K, loc, k, Cm, sh):
    """All points of loc's stream inside interval k, by the definition: partial sums of scaled -ln draws."""
    s = O.prime(K, loc, k)
    pts, T, j = [], 0, 0
    while True:
        j += 1
        T += O.scale(O.neglog(O.draw_time(s, j)), Cm, sh)
        if T >= TWO48:
            return pts
        pts.append((j, T))


def test_next_event_is_first_point_strictly_after(O):
    K = O.key_schedule(99)
    Cm, sh = O.turnover_scale(1.0, 2.0)
    rng = np.random.default_rng(0)
    for loc in range(60):
        k0 = int(rng.integers(0, 1000))
        streams = {k: enumerate_interval(O, K, loc, k, Cm, sh) for k in range(k0, k0 + 40)}
        # queries: fresh, just before/at/after every point, random offsets
        queries = [-1] + [int(v) for v in rng.integers(0, TWO48, 20)]
        for j, T in streams[k0]:
            queries += [T - 1, T, T + 1]
        for f in queries:
            rc, k, j, T, s = O.next_event(K, loc, k0, f, Cm, sh)
            assert rc == 0
            # brute force: first (k', j') in time order with (k', T') > (k0, f)
            exp = None
            for kk in range(k0, k0 + 40):
                for jj, TT in streams[kk]:
                    if kk > k0 or TT > f:
                        exp = (kk, jj, TT); break
                if exp: break
            assert (k, j, T) == exp
            assert s == O.prime(K, loc, k)


def test_alignment_of_parent_and_child(O):
    """L715/L729: any two arrival times with no stream point between them find the same next event."""
    K = O.key_schedule(5)
    Cm, sh = O.turnover_scale(0.8, 2.0)
    rng = np.random.default_rng(1)
    for loc in range(200):
        pts = enumerate_interval(O, K, loc, 7, Cm, sh)
        bounds = [-1] + [T for _, T in pts] + [TWO48 - 1]
        for a, b in zip(bounds[:-1], bounds[1:]):
            if b - a < 3:
                continue
            f1, f2 = sorted(int(v) for v in rng.integers(a + 1, b, 2)) if a >= 0 else (-1, int(rng.integers(0, b)))
            r1 = O.next_event(K, loc, 7, f1, Cm, sh)
            r2 = O.next_event(K, loc, 7, f2, Cm, sh)
            assert r1 == r2


def test_repeated_next_enumerates_ordinals(O):
    K = O.key_schedule(3)
    Cm, sh = O.turnover_scale(1.3, 2.0)
    for loc in range(100):
        k, f, seq = 0, -1, []
        for _ in range(30):
            rc, k2, j, T, _ = O.next_event(K, loc, k, f, Cm, sh)
            seq.append((k2, j, T)); k, f = k2, T
        # inside one interval ordinals are 1,2,3,...; times strictly increase
        for a, b in zip(seq[:-1], seq[1:]):
            assert (b[0], b[2]) > (a[0], a[2])
            assert b[1] == (a[1] + 1 if b[0] == a[0] else 1)


def test_horizon_stop(O):
    K = O.key_schedule(3)
    Cm, sh = O.turnover_scale(1.0, 2.0)
    for loc in range(50):
        rc, k, j, T, _ = O.next_event(K, loc, 0, -1, Cm, sh)
        rc2, k2, _, _, _ = O.next_event(K, loc, 0, -1, Cm, sh, k_stop=k)   # horizon exactly at the event's interval
        if k == 0:
            assert (rc2, k2) == (1, 0)
        else:
            assert (rc2, k2) == (1, k)
        rc3, k3, j3, T3, _ = O.next_event(K, loc, 0, -1, Cm, sh, k_stop=k + 1)
        assert (rc3, k3, j3, T3) == (0, k, j, T)


def test_turnover_times_are_exponential(O):
    """L1206: inter-event times of a lineage that stays put are Exp(lambda). Fisher-combined KS (L1202)."""
    ps = []
    for rep, (lam, dt) in enumerate([(1.0, 2.0), (0.5, 2.0), (1.5, 2.0), (1.0, 3.0), (0.2, 1.0), (4.0, 2.0)]):
        Cm, sh = O.turnover_scale(lam, dt)
        n = 4000
        loc = np.arange(n, dtype=np.uint32) + 1000 * rep
        k = np.zeros(n, np.uint32); f = np.full(n, -1, np.int64)
        t_prev = np.zeros(n)
        gaps = []
        for step in range(12):
            k, j, T, rc = O.batch_next_event(77 + rep, loc, k, f, Cm, sh)
            assert (rc == 0).all()
            t = (k.astype(np.float64) + T / 2.0 ** 48) * dt
            gaps.append(t - t_prev); t_prev = t; f = T.astype(np.int64)
        gaps = np.concatenate(gaps)
        assert (gaps > 0).all()
        ps.append(stats.kstest(gaps * lam, "expon").pvalue)
        assert abs(gaps.mean() * lam - 1.0) < 0.02
    assert min(ps) > 1e-4
    assert stats.combine_pvalues(ps, method="fisher")[1] > 1e-3


def test_points_per_interval_are_poisson(O):
    """L312, L735: N ~ Poi(lambda * dt) points fall into a repriming interval."""
    K = O.key_schedule(1234)
    for lam, dt in ((1.0, 2.0), (0.4, 2.0)):
        Cm, sh = O.turnover_scale(lam, dt)
        counts = np.array([len(enumerate_interval(O, K, loc, 3, Cm, sh)) for loc in range(20000)])
        mu = lam * dt
        kmax = 9
        obs = np.bincount(np.minimum(counts, kmax), minlength=kmax + 1)
        pm = stats.poisson.pmf(np.arange(kmax), mu); exp = np.append(pm, 1 - pm.sum()) * len(counts)
        assert stats.chisquare(obs, exp).pvalue > 1e-3
        assert abs(counts.mean() - mu) < 0.04


def test_points_uniform_inside_interval(O):
    """L310-314: given N, the points of a homogeneous Poisson process are uniform in the interval."""
    K = O.key_schedule(8)
    Cm, sh = O.turnover_scale(1.0, 2.0)
    pts = [T / 2.0 ** 48 for loc in range(15000) for _, T in enumerate_interval(O, K, loc, 11, Cm, sh)]
    assert stats.kstest(pts, "uniform").pvalue > 1e-3


def test_speciation_times_without_dispersal(O):
    """L1208: with dispersal disabled the time to speciation is Exp(lambda * nu); the number of events is
    Geometric(nu). Dispersal is 'disabled' by walking the lineage by hand without moving it."""
    lam, dt, nu = 1.0, 2.0, 0.05
    Cm, sh = O.turnover_scale(lam, dt)
    thr = O.thr(nu)
    n = 6000
    loc = np.arange(n, dtype=np.uint32)
    k = np.zeros(n, np.uint32); f = np.full(n, -1, np.int64)
    alive = np.ones(n, bool); t_spec = np.zeros(n); n_ev = np.zeros(n, int)
    seed = 4242
    while alive.any():
        idx = np.nonzero(alive)[0]
        kk, j, T, rc = O.batch_next_event(seed, loc[idx], k[idx], f[idx], Cm, sh)
        x = O.batch_draw(seed, "spec", loc[idx], kk, j)
        spec = (x >> np.uint64(11)) < np.uint64(thr)
        k[idx] = kk; f[idx] = T.astype(np.int64); n_ev[idx] += 1
        done = idx[spec]
        t_spec[done] = (kk[spec].astype(np.float64) + T[spec] / 2.0 ** 48) * dt
        alive[done] = False
    assert stats.kstest(t_spec * lam * nu, "expon").pvalue > 1e-3
    # Geometric(nu) on {1,2,...}
    assert abs(n_ev.mean() - 1 / nu) < 4 * np.sqrt((1 - nu) / nu ** 2 / n)
    kmax = 60
    obs = np.bincount(np.minimum(n_ev, kmax), minlength=kmax + 1)[1:]
    pm = stats.geom.pmf(np.arange(1, kmax), nu); exp = np.append(pm, 1 - pm.sum()) * n
    assert stats.chisquare(obs, exp).pvalue > 1e-3


def test_bernoulli_threshold(O):
    assert O.thr(0.0) == 0 and O.thr(1.0) == 1 << 53 and O.thr(0.5) == 1 << 52
    assert O.thr(1e-6) == int(np.floor(np.ldexp(1e-6, 53)))
