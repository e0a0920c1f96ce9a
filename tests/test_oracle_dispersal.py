"""P8 -- dispersal sampling of the oracle: alias tables reproduce the
matrix rows, the rounded-Gaussian thresholds reproduce the discretised normal, uniform dispersal visits all
indexed locations equally, and the two samplers agree in distribution."""
import math
import numpy as np
from scipy import stats

NONSPATIAL, SPATIALLY_IMPLICIT, EXPLICIT_MATRIX, EXPLICIT_GAUSSIAN = 0, 1, 2, 3


def pooled_chi2(obs, exp, min_exp=8):
    """chi^2 goodness of fit with all bins of expectation < min_exp pooled into one (dropped if empty)."""
    obs = np.asarray(obs, float); exp = np.asarray(exp, float)
    keep = exp >= min_exp
    o, e = obs[keep], exp[keep]
    if (~keep).any() and exp[~keep].sum() > 0:
        o = np.append(o, obs[~keep].sum()); e = np.append(e, exp[~keep].sum())
    return stats.chisquare(o, e * (o.sum() / e.sum())).pvalue


def alias_mass(th, al):
    n = len(th)
    mass = np.zeros(n)
    for c in range(n):
        acc = th[c] / 2.0 ** 32
        mass[c] += acc / n
        mass[al[c]] += (1.0 - acc) / n
    return mass


def test_alias_row_reconstructs_weights(O):
    rng = np.random.default_rng(0)
    for n in (1, 2, 3, 17, 256, 1000):
        for trial in range(4):
            w = rng.random(n) ** 3
            if trial == 1 and n > 3: w[rng.integers(0, n, n // 2)] = 0.0
            if trial == 2: w[:] = 1.0
            if w.sum() == 0: w[0] = 1.0
            th, al = O.alias_row(w)
            # self-accepting entries use 2^32-1 instead of 2^32: error <= 2^-32 per column
            assert np.abs(alias_mass(th, al) - w / w.sum()).max() < 2.0 ** -31 + 1e-12
            assert np.all(th[w == 0] == 0)          # zero-weight columns are never accepted
            assert np.all(w[al[th < 0xFFFFFFFF]] > 0)


def test_alias_construction_order(O):
    """Hand-worked example of DESIGN.md 2.5 step 3: w = (1, 3, 0, 4), n = 4, S = 8, p = (0.5, 1.5, 0, 2.0).
    small = [0, 2], large = [1, 3]; pop (2, 3): thresh[2] = 0, alias[2] = 3, p[3] = 1.0 -> large;
    pop (0, 3): thresh[0] = 2^31, alias[0] = 3, p[3] = 0.5 -> small; pop (3, 1): thresh[3] = 2^31, alias[3] = 1,
    p[1] = 1.0 -> large; leftover 1: thresh = 2^32-1, alias = 1."""
    th, al = O.alias_row(np.array([1.0, 3.0, 0.0, 4.0]))
    assert list(th) == [1 << 31, 0xFFFFFFFF, 0, 1 << 31]
    assert list(al) == [3, 1, 3, 1]


def test_gauss_table_masses(O):
    for sigma in (0.3, 1.0, 2.0, 3.0, 5.0):
        R, TG = O.gauss_table(sigma)
        assert R == math.ceil(10 * sigma) and len(TG) == 2 * R
        assert np.all(np.diff(TG.astype(np.int64)) >= 0)
        cdf = np.concatenate([[0.0], TG / 2.0 ** 32, [1.0]])
        mass = np.diff(cdf)
        d = np.arange(-R, R + 1)
        exp = stats.norm.cdf((d + 0.5) / sigma) - stats.norm.cdf((d - 0.5) / sigma)
        assert np.abs(mass - exp).max() < 2.0 ** -31
        assert abs(mass @ d) < 1e-6
        if sigma >= 1.0:        # Sheppard's correction holds for sigma >~ 1
            assert abs(mass @ (d * d) - (sigma ** 2 + 1 / 12.0)) < 1e-3 * sigma ** 2
        # lookup = smallest index with u < TG[i]
        for u in (0, 1, int(TG[R]) - 1, int(TG[R]), 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF):
            exp_d = int(np.searchsorted(TG, u, side="right")) - R
            assert O.gauss_lookup(TG, R, u) == exp_d
        assert O.gauss_lookup(TG, R, 0x7FFFFFFF) == 0 and O.gauss_lookup(TG, R, 0x80000000) == 0


def test_gaussian_dispersal_per_axis_chi2(O):
    """L1216: each axis of the dispersal follows the discretised normal (all cells habitat, deme 1)."""
    W = H = 64; sigma = 2.0
    sc = O.Scenario(EXPLICIT_GAUSSIAN, W, H, uniform_deme=1, sigma=sigma, delta_t=2.0)
    n = 200000
    rng = np.random.default_rng(1)
    loc = rng.integers(0, W * H, n).astype(np.uint32)
    out = O.batch_disperse(sc, 9, loc, rng.integers(0, 1000, n).astype(np.uint32), 1)
    dx = (out % W).astype(int) - (loc % W).astype(int); dy = (out // W).astype(int) - (loc // W).astype(int)
    dx = (dx + W // 2) % W - W // 2; dy = (dy + H // 2) % H - H // 2
    d = np.arange(-8, 9)
    exp = stats.norm.cdf((d + 0.5) / sigma) - stats.norm.cdf((d - 0.5) / sigma)
    exp[0] += stats.norm.cdf((-8.5) / sigma); exp[-1] += stats.norm.sf(8.5 / sigma)
    for v in (dx, dy):
        obs = np.bincount(np.clip(v, -8, 8) + 8, minlength=17)
        assert stats.chisquare(obs, exp * n).pvalue > 1e-3
    assert abs(np.corrcoef(dx, dy)[0, 1]) < 0.01


def test_gaussian_resampling_never_lands_on_non_habitat(O):
    W = H = 32
    rng = np.random.default_rng(2)
    deme = (rng.random(W * H) < 0.4).astype(np.uint32) * rng.integers(1, 4, W * H).astype(np.uint32)
    deme[5] = 3
    sc = O.Scenario(EXPLICIT_GAUSSIAN, W, H, deme=deme, sigma=1.5, delta_t=2.0)
    prefix = np.concatenate([[0], np.cumsum(deme)]).astype(np.int64)
    n_ind = int(prefix[-1])
    loc = rng.integers(0, n_ind, 100000).astype(np.uint32)
    out = O.batch_disperse(sc, 3, loc, np.arange(len(loc), dtype=np.uint32), 2)     # distinct events
    assert out.max() < n_ind
    # conditional distribution: target cell ~ kernel restricted to habitat (rejection sampling), index uniform
    cell_of = np.searchsorted(prefix, out, side="right") - 1
    assert np.all(deme[cell_of] > 0)
    idx = out.astype(np.int64) - prefix[cell_of]
    for dsize in (2, 3):
        sel = deme[cell_of] == dsize
        assert stats.chisquare(np.bincount(idx[sel], minlength=dsize)).pvalue > 1e-3
    # one origin cell in detail
    origin = int(np.flatnonzero(deme)[10]); x0, y0 = origin % W, origin // W
    locs = np.full(150000, prefix[origin], np.uint32)
    out = O.batch_disperse(sc, 4, locs, np.arange(150000, dtype=np.uint32), 1)
    cells = np.searchsorted(prefix, out, side="right") - 1
    R, TG = O.gauss_table(1.5)
    mass1 = np.diff(np.concatenate([[0.0], TG / 2.0 ** 32, [1.0]]))
    exp = np.zeros(W * H)
    for dy in range(-R, R + 1):
        for dx in range(-R, R + 1):
            c = ((y0 + dy) % H) * W + (x0 + dx) % W
            exp[c] += mass1[dx + R] * mass1[dy + R]
    exp[deme == 0] = 0; exp /= exp.sum()
    assert pooled_chi2(np.bincount(cells, minlength=W * H), exp * len(out)) > 1e-3


def test_matrix_dispersal_matches_rows(O):
    from paper_2108_05815_b200 import inputs as I
    W = H = 6; deme = 3
    M = I.torus_gaussian_matrix(W, H, 1.0)
    sc = O.Scenario(EXPLICIT_MATRIX, W, H, uniform_deme=deme, matrix=M, delta_t=2.0)
    th, al = sc.alias_tables()
    for row in (0, 7, 35):
        t2, a2 = O.alias_row(M[row])
        assert (th[row] == t2).all() and (al[row] == a2).all()
        n = 120000
        out = O.batch_disperse(sc, 6, np.full(n, row * deme + 1, np.uint32), np.arange(n, dtype=np.uint32), 1)
        cells = out // deme
        assert pooled_chi2(np.bincount(cells, minlength=W * H), M[row] * n) > 1e-3
        assert stats.chisquare(np.bincount(out % deme, minlength=deme)).pvalue > 1e-3


def test_alias_vs_gauss_sampler_cross_check(O):
    """A matrix built from the rounded-Gaussian masses (wrapped on the torus) sampled by alias tables gives the
    same target distribution as the threshold-table sampler."""
    W = H = 32; sigma = 1.0
    R, TG = O.gauss_table(sigma)
    m1 = np.diff(np.concatenate([[0.0], TG / 2.0 ** 32, [1.0]]))
    k1 = np.zeros(W)
    for d in range(-R, R + 1): k1[d % W] += m1[d + R]
    sc_g = O.Scenario(EXPLICIT_GAUSSIAN, W, H, uniform_deme=1, sigma=sigma, delta_t=2.0)
    xs = np.arange(W)
    Mx = k1[(xs[None, :] - xs[:, None]) % W]
    M = (Mx[:, None, :, None] * Mx[None, :, None, :]).reshape(W * H, W * H)
    sc_m = O.Scenario(EXPLICIT_MATRIX, W, H, uniform_deme=1, matrix=M, delta_t=2.0)
    n = 100000; origin = 5 * W + 7
    og = O.batch_disperse(sc_g, 1, np.full(n, origin, np.uint32), np.arange(n, dtype=np.uint32), 1)
    om = O.batch_disperse(sc_m, 2, np.full(n, origin, np.uint32), np.arange(n, dtype=np.uint32), 1)
    a = np.bincount(og, minlength=W * H); b = np.bincount(om, minlength=W * H)
    keep = (a + b) > 20
    assert stats.chi2_contingency(np.vstack([np.append(a[keep], a[~keep].sum() + 1), np.append(b[keep], b[~keep].sum() + 1)]))[1] > 1e-3


def test_uniform_dispersal_visits_all_locations_equally(O):
    """L1212: non-spatial dispersal is uniform over all indexed locations (self included, R12)."""
    J = 997
    sc = O.Scenario(NONSPATIAL, 1, 1, uniform_deme=J, delta_t=2.0)
    n = 300000
    out = O.batch_disperse(sc, 8, np.arange(n, dtype=np.uint32) % J, np.arange(n, dtype=np.uint32) // J, 1)
    assert out.max() == J - 1
    assert stats.chisquare(np.bincount(out, minlength=J)).pvalue > 1e-3
    assert abs((out == (np.arange(n) % J)).mean() - 1.0 / J) < 4 * np.sqrt(1.0 / J / n)


def test_implicit_dispersal(O):
    Jl, Jm, m = 1000, 5000, 0.25
    sc = O.Scenario(SPATIALLY_IMPLICIT, local_size=Jl, meta_size=Jm, migration=m, delta_t=2.0)
    n = 200000
    out = O.batch_disperse(sc, 8, np.arange(n, dtype=np.uint32) % Jl, np.arange(n, dtype=np.uint32) // Jl, 1)
    mig = out >= Jl
    assert abs(mig.mean() - m) < 4 * np.sqrt(m * (1 - m) / n)
    assert stats.chisquare(np.bincount(out[~mig], minlength=Jl)).pvalue > 1e-3
    assert stats.chisquare(np.bincount(out[mig] - Jl, minlength=Jm)).pvalue > 1e-3
    out2 = O.batch_disperse(sc, 8, Jl + (np.arange(n, dtype=np.uint32) % Jm), 3, 1)
    assert out2.min() >= Jl and out2.max() < Jl + Jm          # no return migration (R13)


def test_scenario_validation(O):
    import pytest
    with pytest.raises(ValueError):
        O.Scenario(EXPLICIT_GAUSSIAN, 8, 8, uniform_deme=1, sigma=1.0)        # R = 10 >= 8
    with pytest.raises(ValueError):
        O.Scenario(NONSPATIAL, 2, 1, uniform_deme=5)
    with pytest.raises(ValueError):
        O.Scenario(EXPLICIT_MATRIX, 2, 2, deme=np.array([1, 0, 1, 1], np.uint32), matrix=np.ones((4, 4)))
    with pytest.raises(ValueError):
        O.Scenario(NONSPATIAL, 1, 1, uniform_deme=5, uniform_turnover=1.0, delta_t=1000.0)
