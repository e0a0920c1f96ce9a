"""P2 -- the oracle's fixed-point -ln (PAPER.md Eq. C.3) against an
independent 60-digit logarithm (mpmath), plus monotonicity, edge cases and frozen vectors."""
import os
import numpy as np
import mpmath

HERE = os.path.dirname(os.path.abspath(__file__))
BOUND = 2.0 ** -43


def exact_neglog(x):
    """-ln(U), U = M * 2^-(z+50) with M the 50-bit odd mantissa of DESIGN.md 2.3 (definition, not the algorithm)."""
    z = 64 - x.bit_length()
    y = (x << z) & ((1 << 64) - 1)
    M = (y >> 14) | 1
    return -(mpmath.log(mpmath.mpf(M)) - (z + 50) * mpmath.log(2))


def test_against_high_precision_log(O):
    mpmath.mp.dps = 60
    rng = np.random.default_rng(3)
    xs = [int(v) for v in rng.integers(0, 1 << 64, 20000, dtype=np.uint64)]
    xs += [int(v) >> int(s) for v, s in zip(rng.integers(0, 1 << 64, 4000, dtype=np.uint64), rng.integers(0, 64, 4000))]
    xs += [1, 2, 3, (1 << 64) - 1, (1 << 64) - 2, 1 << 63, (1 << 63) - 1, (1 << 63) + 1]
    xs += [(1 << b) + d for b in range(1, 64) for d in (-1, 0, 1)]
    # table-bin boundaries: mantissa just below / at a multiple of 2^-9
    xs += [((512 + i) << 54) + d for i in range(0, 512, 7) for d in (-1, 0, 1) if 0 < ((512 + i) << 54) + d < (1 << 64)]
    xs = [x for x in xs if x != 0]          # x = 0 is not normalised; pinned in test_zero_and_extremes
    got = O.batch_neglog(np.array(xs, dtype=np.uint64))
    worst = 0.0
    for x, e in zip(xs, got):
        err = abs(mpmath.mpf(int(e)) / mpmath.mpf(2) ** 56 - exact_neglog(x))
        worst = max(worst, float(err))
    assert worst <= BOUND, worst


def test_mantissa_granularity_is_negligible(O):
    """U = (x + 1/2)/2^64 differs from M*2^-(z+50) by at most 2^-49 relative: -ln agrees to 2^-48."""
    mpmath.mp.dps = 60
    rng = np.random.default_rng(4)
    for x in [int(v) for v in rng.integers(1 << 20, 1 << 64, 2000, dtype=np.uint64)]:
        true = -mpmath.log((mpmath.mpf(x) + 0.5) / mpmath.mpf(2) ** 64)
        assert abs(true - exact_neglog(x)) < mpmath.mpf(2) ** -48


def test_zero_and_extremes(O):
    LN2_56 = 49946518145322873
    assert O.neglog(0) == 65 * LN2_56 - 128            # DESIGN.md section 3 ("x = 0 needs no special case")
    assert O.neglog((1 << 64) - 1) < 2 ** 10           # U -> 1: -ln U -> 2^-50
    assert abs(O.neglog(1 << 63) / 2.0 ** 56 - np.log(2.0)) < 1e-12


def test_monotone_up_to_bound(O):
    rng = np.random.default_rng(6)
    x = np.sort(rng.integers(0, 1 << 64, 200000, dtype=np.uint64))
    e = O.batch_neglog(x).astype(np.int64)
    viol = (e[1:] - e[:-1]).max()          # must be non-increasing up to the error bound
    assert viol <= int(2 * BOUND * 2 ** 56)
    # dense scan across several table-bin boundaries at full resolution of M (step 2^14 in y)
    base = (512 + 37) << 54
    xs = np.uint64(base) + (np.arange(-3000, 3000, dtype=np.int64) * (1 << 14)).astype(np.uint64)
    e = O.batch_neglog(xs).astype(np.int64)
    assert (e[1:] - e[:-1]).max() <= int(2 * BOUND * 2 ** 56)


def test_exponential_distribution_of_neglog_of_draws(O):
    from scipy import stats
    n = 400000
    x = O.batch_draw(11, "time", np.arange(n, dtype=np.uint32), 0, 1)
    e = O.batch_neglog(x) / 2.0 ** 56
    assert stats.kstest(e, "expon").pvalue > 1e-3
    assert abs(e.mean() - 1.0) < 0.01 and abs(e.var() - 1.0) < 0.02


def test_scale_and_turnover_scale(O):
    Cm, sh = O.turnover_scale(1.0, 2.0)
    assert (Cm, sh) == (1 << 31, 8)
    E = O.neglog(123456789123456789)
    assert O.scale(E, Cm, sh) == E >> 9                 # E/2 in Q16.48 = E * 2^-1 * 2^-8
    for lam, dt in ((0.5, 2.0), (1.5, 2.0), (0.731, 3.0), (0.01, 2.0), (20.0, 3.0)):
        Cm, sh = O.turnover_scale(lam, dt)
        assert (1 << 31) <= Cm < (1 << 32)
        inv = Cm * 2.0 ** (-31 + 7 - sh)
        assert abs(inv * lam * dt - 1.0) < 2.0 ** -30
        import fractions
        exact = fractions.Fraction(E) * Cm / (1 << 32) / (1 << sh)
        assert O.scale(E, Cm, sh) == int(exact)         # bits of the exact product, truncated
    import pytest
    with pytest.raises(ValueError):
        O.turnover_scale(1.0, 1000.0)


def test_time_conversion(O):
    assert O.time_of(0, 0, 2.0) == 0.0
    assert O.time_of(3, 1 << 47, 2.0) == 7.0
    assert O.time_of(5, 1 << 46, 3.0) == 15.75


def test_golden_vectors(O):
    for line in open(os.path.join(HERE, "golden", "neglog_vectors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        x, v = line.split()
        assert O.neglog(int(x, 16)) == int(v)


def test_table_matches_definition():
    """Q[i] = ceil(2^21/(512+i)), A[i] = round(-ln(Q/4096) 2^56): recompute with mpmath (not the generator's decimal)."""
    mpmath.mp.dps = 70
    rows = []
    for line in open(os.path.join(os.path.dirname(HERE), "oracle", "neglog_table.inc")):
        if line.startswith("{"):
            q, a = line.strip().rstrip(",").strip("{}").split(",")
            rows.append((int(q.strip().rstrip("u")), int(a.strip().rstrip("ul"))))
    assert len(rows) == 512
    for i, (q, a) in enumerate(rows):
        assert q == -((-(1 << 21)) // (512 + i))
        assert a == int(mpmath.nint(-mpmath.log(mpmath.mpf(q) / 4096) * mpmath.mpf(2) ** 56))
