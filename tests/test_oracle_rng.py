"""P1 -- pins for the primeable hash RNG of the oracle (PAPER.md 5.2.1 L693-707,
avalanche criteria L351-355, correlation check L1198). The bit values themselves are "parity
unpinned" against the paper (different mixer, R2); golden vectors guard regressions."""
import os
import numpy as np
from scipy import stats

HERE = os.path.dirname(os.path.abspath(__file__))


def _bit_flip_probs(f, x, bit):
    d = f(x) ^ f(x ^ np.uint64(1 << bit))
    bits = np.unpackbits(d.view(np.uint8).reshape(-1, 8), axis=1, bitorder="little")
    return bits.mean(axis=0)


def test_F_is_a_bijection_on_samples_and_avalanches(O):
    rng = np.random.default_rng(1)
    N = 1 << 17
    x = rng.integers(0, 1 << 64, N, dtype=np.uint64)
    assert len(np.unique(O.batch_F(x))) == len(np.unique(x))
    worst = 0.0
    for bit in range(64):
        p = _bit_flip_probs(O.batch_F, x, bit)
        worst = max(worst, np.abs(p - 0.5).max())
    assert worst < 0.01          # strict avalanche criterion, L351-355 (noise sd here is 0.0014)


def test_F_avalanches_on_sequential_counters(O):
    x = np.arange(1 << 17, dtype=np.uint64)
    worst = max(np.abs(_bit_flip_probs(O.batch_F, x, b) - 0.5).max() for b in range(20))
    assert worst < 0.01


def test_draw_avalanche_over_seed_loc_k_j(O):
    """Flip every input bit of (seed, loc, k, j): each output bit of the time draw flips w.p. 1/2."""
    rng = np.random.default_rng(2)
    N = 1 << 15
    loc = rng.integers(0, 1 << 22, N, dtype=np.uint32)      # structured, small inputs
    k = rng.integers(0, 1 << 10, N, dtype=np.uint32)
    j = rng.integers(1, 8, N, dtype=np.uint32)
    seed = 42
    base = O.batch_draw(seed, "time", loc, k, j)

    def dev(other):
        d = base ^ other
        bits = np.unpackbits(d.view(np.uint8).reshape(-1, 8), axis=1, bitorder="little")
        return np.abs(bits.mean(axis=0) - 0.5).max()
    worst = 0.0
    for b in range(32):
        worst = max(worst, dev(O.batch_draw(seed, "time", loc ^ np.uint32(1 << b), k, j)))
        worst = max(worst, dev(O.batch_draw(seed, "time", loc, k ^ np.uint32(1 << b), j)))
    for b in range(12):
        worst = max(worst, dev(O.batch_draw(seed, "time", loc, k, j ^ np.uint32(1 << b))))
    for b in range(64):
        worst = max(worst, dev(O.batch_draw(seed ^ (1 << b), "time", loc, k, j)))
    assert worst < 0.02          # noise sd 0.0028 at N = 2^15; 172 x 64 cells


def test_lanes_are_distinct_and_uncorrelated(O):
    n = 200000
    loc = np.arange(n, dtype=np.uint32)
    lanes = {ln: O.batch_draw(7, ln, loc, 3, 2) for ln in ("time", "spec", "disp", "index", "migr")}
    names = list(lanes)
    for a in range(len(names)):
        for b in range(a + 1, len(names)):
            xa, xb = lanes[names[a]], lanes[names[b]]
            assert not np.any(xa == xb)
            rho, _ = stats.spearmanr(xa[:20000].astype(np.float64), xb[:20000].astype(np.float64))
            assert abs(rho) < 0.03
    # resample attempts differ from each other
    d0 = O.batch_draw(7, "disp", loc, 3, 2, r=0); d1 = O.batch_draw(7, "disp", loc, 3, 2, r=1)
    assert not np.any(d0 == d1)


def test_uniformity_chi2_of_bytes(O):
    n = 1 << 20
    x = O.batch_draw(5, "time", np.arange(n, dtype=np.uint32) % 4099, np.arange(n, dtype=np.uint32) // 4099, 1)
    for shift in (56, 32, 24, 0):
        counts = np.bincount(((x >> np.uint64(shift)) & np.uint64(255)).astype(np.int64), minlength=256)
        assert stats.chisquare(counts).pvalue > 1e-4


def test_adjacent_streams_uncorrelated(O):
    """streams of individuals starting at adjacent locations show no Spearman correlation."""
    js = np.arange(1, 101, dtype=np.uint32)
    ps = []
    for seed in range(200):
        streams = [O.batch_draw(seed, "time", np.full(100, loc, np.uint32), 0, js).astype(np.float64) for loc in (0, 1, 2, 3)]
        for a in range(4):
            for b in range(a + 1, 4):
                ps.append(stats.spearmanr(streams[a], streams[b]).pvalue)
    ps = np.array(ps)
    # p-values of independent streams are uniform: KS against U(0,1)
    assert stats.kstest(ps, "uniform").pvalue > 1e-3
    assert (ps < 0.001).mean() < 0.01


def test_golden_vectors(O):
    """Frozen outputs written by tests/golden/gen_golden.py (calls oracle/ only): regression guard."""
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "rng_vectors.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) >= 40
    for seed, lane, loc, k, j, r, val in rows:
        got = O.batch_draw(int(seed), lane, np.array([int(loc)], np.uint32), int(k), int(j), r=int(r))[0]
        assert int(got) == int(val, 16), (seed, lane, loc, k, j, r)


def test_key_schedule_depends_on_seed(O):
    ks = np.array([O.key_schedule(s) for s in range(64)])
    assert len({tuple(r) for r in ks}) == 64
    assert O.prime(O.key_schedule(1), 5, 6) != O.prime(O.key_schedule(2), 5, 6)
