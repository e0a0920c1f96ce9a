"""P5-P7 -- whole-model pins of the oracle.
P5: Ewens sampling formula for the non-spatial model (PAPER.md Eq. B.1) and tiny-J closed forms.
P6: species-abundance distribution against the classical event-by-event coalescence (App. G.3).
P7: spatially implicit species richness against Eq. B.4 (L1839), weak."""
import os
import numpy as np
from scipy import stats
from scipy.special import digamma, gammaln

from classical import simulate_classical, sad_of

HERE = os.path.dirname(os.path.abspath(__file__))
NONSPATIAL, SPATIALLY_IMPLICIT, EXPLICIT_MATRIX, EXPLICIT_GAUSSIAN = 0, 1, 2, 3


def ewens_S(J, nu, self_replacement=True):
    theta = (J if self_replacement else J - 1) * nu / (1 - nu)      # footnote L1816
    return theta * (digamma(theta + J) - digamma(theta)), theta


def test_paper_formula_values():
    """golden/ewens.txt holds the numbers derived from Eq. B.1 for config 1."""
    vals = dict(l.split("=") for l in open(os.path.join(HERE, "golden", "ewens.txt")) if "=" in l and not l.startswith("#"))
    S, theta = ewens_S(10_000, 1e-3)
    assert abs(S - float(vals["E_S_C1"])) < 1e-3 and abs(theta - float(vals["theta_C1"])) < 1e-5
    S2, _ = ewens_S(10_000, 1e-3, self_replacement=False)
    assert abs(S2 - float(vals["E_S_C1_no_self"])) < 1e-3


def test_ewens_mean_config1(O):
    """configs[0]: J = 1e4, nu = 1e-3, 100 seeds: mean richness within 3 s.e. of 69.65 (sd 7.69)."""
    sc = O.Scenario(NONSPATIAL, 1, 1, uniform_deme=10_000, delta_t=2.0)
    res = [sc.simulate(seed, 1e-3) for seed in range(100)]
    S = np.array([r["richness"] for r in res])
    exp, theta = ewens_S(10_000, 1e-3)
    # Var[S] = sum_i theta*i/(theta+i)^2
    i = np.arange(10_000)
    sd = np.sqrt((theta * i / (theta + i) ** 2).sum())
    assert abs(S.mean() - exp) < 3 * sd / 10
    assert 0.75 * sd < S.std(ddof=1) < 1.25 * sd
    # every unique event is a speciation w.p. nu  =>  E[#unique events] = E[S]/nu
    ev = np.array([r["stats"]["n_events"] for r in res])
    assert abs(ev.mean() - exp / 1e-3) < 3 * (sd / 1e-3) / 10 + 3 * np.sqrt(exp / 1e-3 / 1e-3) / 10
    # labels are a partition of the sample; abundances add up
    for r in res[:5]:
        assert r["events"]["abundance"].sum() == 10_000
        assert (np.bincount(r["labels"], minlength=r["richness"]) == r["events"]["abundance"]).all()


def test_ewens_abundance_spectrum(O):
    """E[phi_a] = (theta/a) J!/(J-a)! Gamma(theta+J-a)/Gamma(theta+J) (Ewens; textbook)."""
    J, nu, nseeds = 400, 0.02, 1500
    sc = O.Scenario(NONSPATIAL, 1, 1, uniform_deme=J, delta_t=2.0)
    theta = J * nu / (1 - nu)
    phi = np.zeros(J + 1)
    for seed in range(nseeds):
        ab = sc.simulate(1000 + seed, nu)["events"]["abundance"]
        phi += np.bincount(ab, minlength=J + 1)
    phi /= nseeds
    a = np.arange(1, 9)
    exp = theta / a * np.exp(gammaln(J + 1) - gammaln(J - a + 1) + gammaln(theta + J - a) - gammaln(theta + J))
    # phi_a are sums of many weakly dependent indicators: use a 5 sigma Poisson-like band
    assert np.all(np.abs(phi[1:9] - exp) < 5 * np.sqrt(exp / nseeds) + 0.01)


def test_tiny_J_closed_forms(O):
    """E[S] = sum_{i<J} theta/(theta+i), theta = J nu/(1-nu): self-replacement allowed (R12). The values under
    the other convention (theta = (J-1)nu/(1-nu)) are far outside the acceptance band."""
    for J, nu, exp, other in ((2, 0.5, 1.666667, 1.5), (3, 0.5, 2.35, 2.166667), (4, 0.1, 1.618543, 1.466), (8, 0.5, 5.802975, 5.62)):
        theta = J * nu / (1 - nu)
        assert abs(sum(theta / (theta + i) for i in range(J)) - exp) < 1e-4
        sc = O.Scenario(NONSPATIAL, 1, 1, uniform_deme=J, delta_t=2.0)
        n = 40000
        S = np.array([sc.simulate(seed, nu)["richness"] for seed in range(n)])
        se = S.std(ddof=1) / np.sqrt(n)
        assert abs(S.mean() - exp) < 4 * se, (J, nu, S.mean(), exp)
        assert abs(S.mean() - other) > 6 * se


def _compare_sad(oracle_sads, classical_sads, maxa):
    """chi^2 homogeneity test on pooled abundance-class counts + KS on richness."""
    a = np.zeros(maxa + 1); b = np.zeros(maxa + 1)
    for s in oracle_sads:
        s = np.asarray(s); a[: min(len(s), maxa)] += s[:maxa]; a[maxa] += s[maxa:].sum()
    for s in classical_sads:
        s = np.asarray(s); b[: min(len(s), maxa)] += s[:maxa]; b[maxa] += s[maxa:].sum()
    keep = (a + b) > 10
    chi = stats.chi2_contingency(np.vstack([a[keep], b[keep]]))
    return chi[1]


def test_sad_vs_classical_nonspatial(O):
    J, nu, n = 24, 0.08, 3000
    sc = O.Scenario(NONSPATIAL, 1, 1, uniform_deme=J, delta_t=2.0)
    o_sads, o_S = [], []
    for seed in range(n):
        r = sc.simulate(seed, nu); o_sads.append(np.bincount(r["events"]["abundance"])); o_S.append(r["richness"])
    rng = np.random.default_rng(1)
    c_sads, c_S = [], []
    for _ in range(n):
        lab = simulate_classical(rng, list(range(J)), lambda l: nu, lambda g, l: int(g.integers(J)))
        c_sads.append(sad_of(lab)); c_S.append(len(set(lab)))
    assert _compare_sad(o_sads, c_sads, 12) > 1e-3
    assert stats.ks_2samp(o_S, c_S).pvalue > 1e-3
    assert abs(np.mean(o_S) - np.mean(c_S)) < 4 * np.sqrt(np.var(o_S) / n + np.var(c_S) / n)


def test_sad_vs_classical_matrix_torus(O):
    """4x4 torus, deme 2, dispersal matrix sampled through the oracle's alias tables vs. direct sampling of the rows."""
    from paper_2108_05815_b200 import inputs as I
    W = H = 4; deme = 2; nu = 0.1; n = 2500
    M = I.torus_gaussian_matrix(W, H, 0.8)
    sc = O.Scenario(EXPLICIT_MATRIX, W, H, uniform_deme=deme, matrix=M, delta_t=2.0)
    o_sads, o_S = [], []
    for seed in range(n):
        r = sc.simulate(seed, nu); o_sads.append(np.bincount(r["events"]["abundance"])); o_S.append(r["richness"])
    rng = np.random.default_rng(2)
    cum = np.cumsum(M, axis=1)

    def disperse(g, l):
        cell, _ = l
        c2 = int(np.searchsorted(cum[cell], g.random() * cum[cell, -1], side="right"))
        return (min(c2, W * H - 1), int(g.integers(deme)))
    starts = [(c, i) for c in range(W * H) for i in range(deme)]
    c_sads, c_S = [], []
    for _ in range(n):
        lab = simulate_classical(rng, starts, lambda l: nu, disperse)
        c_sads.append(sad_of(lab)); c_S.append(len(set(lab)))
    assert _compare_sad(o_sads, c_sads, 12) > 1e-3
    assert stats.ks_2samp(o_S, c_S).pvalue > 1e-3


def test_sad_vs_classical_gaussian_habitat_turnover(O):
    """8x8 torus with holes, demes 1-3, per-cell turnover, rounded Gaussian with resampling off non-habitat."""
    W = H = 8; nu = 0.08; sigma = 0.3; n = 2500        # R = ceil(10 sigma) = 3 < 8
    rng0 = np.random.default_rng(5)
    deme = rng0.integers(0, 4, W * H).astype(np.uint32)
    deme[0] = 2
    turnover = 0.5 + rng0.random(W * H)
    sc = O.Scenario(EXPLICIT_GAUSSIAN, W, H, deme=deme, turnover=turnover, sigma=sigma, delta_t=2.0)
    o_sads, o_S = [], []
    for seed in range(n):
        r = sc.simulate(seed, nu); o_sads.append(np.bincount(r["events"]["abundance"])); o_S.append(r["richness"])
    rng = np.random.default_rng(3)

    def disperse(g, l):
        cell, _ = l
        x0, y0 = cell % W, cell // W
        while True:
            dx = int(np.rint(g.normal(0.0, sigma))); dy = int(np.rint(g.normal(0.0, sigma)))
            c2 = ((y0 + dy) % H) * W + (x0 + dx) % W
            if deme[c2] > 0:
                return (c2, int(g.integers(deme[c2])))

    class Rate:
        max = float(turnover.max())
        def __call__(self, l): return float(turnover[l[0]])
    starts = [(c, i) for c in range(W * H) for i in range(deme[c])]
    c_sads, c_S = [], []
    for _ in range(n):
        lab = simulate_classical(rng, starts, lambda l: nu, disperse, rate_of=Rate())
        c_sads.append(sad_of(lab)); c_S.append(len(set(lab)))
    assert _compare_sad(o_sads, c_sads, 12) > 1e-3
    assert stats.ks_2samp(o_S, c_S).pvalue > 1e-3
    assert abs(np.mean(o_S) - np.mean(c_S)) < 4 * np.sqrt(np.var(o_S) / n + np.var(c_S) / n)


def test_sad_vs_classical_implicit(O):
    Jl, Jm, m, nu, n = 12, 40, 0.3, 0.1, 3000
    sc = O.Scenario(SPATIALLY_IMPLICIT, local_size=Jl, meta_size=Jm, migration=m, delta_t=2.0)
    o_sads, o_S = [], []
    for seed in range(n):
        r = sc.simulate(seed, nu); o_sads.append(np.bincount(r["events"]["abundance"])); o_S.append(r["richness"])
    rng = np.random.default_rng(4)

    def disperse(g, l):
        if l < Jl and g.random() >= m:
            return int(g.integers(Jl))
        return Jl + int(g.integers(Jm))
    c_sads, c_S = [], []
    for _ in range(n):
        lab = simulate_classical(rng, list(range(Jl)), lambda l: nu if l >= Jl else 0.0, disperse)
        c_sads.append(sad_of(lab)); c_S.append(len(set(lab)))
    assert _compare_sad(o_sads, c_sads, 8) > 1e-3
    assert stats.ks_2samp(o_S, c_S).pvalue > 1e-3


def test_spatially_implicit_formula_B4(O):
    """Weak pin (P7): Eq. B.4 (L1839) with a large metacommunity; accept within 4 % over 12 seeds."""
    Jl, Jm, m, nu = 20_000, 1_000_000, 0.01, 1e-3
    gamma = (Jl - 1) * m / (1 - m)
    theta = (Jm - 1) * nu / (1 - nu)
    immigrants = gamma * (digamma(gamma + Jl) - digamma(gamma))
    exp = theta * (digamma(theta + immigrants) - digamma(theta))
    sc = O.Scenario(SPATIALLY_IMPLICIT, local_size=Jl, meta_size=Jm, migration=m, delta_t=2.0)
    S = np.array([sc.simulate(seed, nu)["richness"] for seed in range(12)])
    assert abs(S.mean() / exp - 1.0) < 0.04, (S.mean(), exp)
