"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the oracle tests, the GPU parity tests and bench.py. It holds NO arithmetic
of the method (no hashing, no sampling of events): only numpy recipes that produce the landscapes
(habitat, turnover, dispersal matrix, sample mask) standing in for the paper's Madingley maps
(PAPER.md L1334, L1443), which are not available.

Every config is a plain dict:
  kind, width, height, deme (u32[ncells] or None), uniform_deme, turnover (f64[ncells] or None),
  uniform_turnover, matrix (f64[ncells, ncells] or None), sigma, local_size, meta_size, migration,
  delta_t, sampler (0 exponential, 1 Poisson event-time sampler), nu, seed, mask (u8[n_individuals] or None), name
"""
import math
import numpy as np

NONSPATIAL, SPATIALLY_IMPLICIT, EXPLICIT_MATRIX, EXPLICIT_GAUSSIAN = 0, 1, 2, 3


def _base(name, kind, **kw):
    cfg = dict(name=name, kind=kind, width=1, height=1, deme=None, uniform_deme=0, turnover=None,
               uniform_turnover=1.0, matrix=None, sigma=0.0, local_size=0, meta_size=0, migration=0.0,
               delta_t=2.0, nu=1e-3, seed=42, mask=None, sampler=0, past_deme=None, past_start_k=None)
    cfg.update(kw)
    return cfg


def c1_nonspatial(J=10_000, nu=1e-3, seed=42):
    """configs[0]: non-spatial Moran community, all sampled."""
    return _base("C1-nonspatial-J%d" % J, NONSPATIAL, uniform_deme=J, nu=nu, seed=seed)


def c2_implicit(J_local=100_000, J_meta=1_000_000_000, m=0.01, nu=1e-4, seed=42):
    """configs[1]: spatially implicit, dynamic finite metacommunity."""
    return _base("C2-implicit-Jl%d-Jm%d" % (J_local, J_meta), SPATIALLY_IMPLICIT, local_size=J_local,
                 meta_size=J_meta, migration=m, nu=nu, seed=seed)


def _phi(z):
    return 0.5 * (1.0 + math.erf(z / math.sqrt(2.0)))


def torus_gaussian_matrix(width, height, sigma):
    """Row-normalised dispersal matrix: discretised Gaussian summed over periodic images."""
    def axis_kernel(n):
        k = np.zeros(n)
        for d in range(n):
            tot = 0.0
            for img in range(-8, 9):
                dd = d + img * n
                if abs(dd) > 12 * sigma + n:
                    continue
                tot += _phi((dd + 0.5) / sigma) - _phi((dd - 0.5) / sigma)
            k[d] = tot
        return k
    kx, ky = axis_kernel(width), axis_kernel(height)
    xs = np.arange(width)
    ys = np.arange(height)
    Mx = kx[(xs[None, :] - xs[:, None]) % width]        # [x, x']
    My = ky[(ys[None, :] - ys[:, None]) % height]       # [y, y']
    M = (My[:, None, :, None] * Mx[None, :, None, :]).reshape(width * height, width * height)
    M /= M.sum(axis=1, keepdims=True)
    return np.ascontiguousarray(M)


def c3_matrix(side=64, deme=10, sigma=2.0, nu=1e-4, seed=42):
    """configs[2]: spatially explicit torus, per-cell dispersal matrix sampled by alias tables."""
    return _base("C3-matrix-%dx%d" % (side, side), EXPLICIT_MATRIX, width=side, height=side, uniform_deme=deme,
                 matrix=torus_gaussian_matrix(side, side, sigma), sigma=sigma, nu=nu, seed=seed)


def c4_gaussian(side=1000, p_habitat=0.7, sigma=3.0, nu=1e-5, seed=42, map_seed=1, turnover_seed=2):
    """configs[3]: i.i.d. habitat p=0.7, deme 1, per-cell turnover U[0.5,1.5), rounded Gaussian dispersal."""
    rng = np.random.Generator(np.random.PCG64(map_seed))
    deme = (rng.random(side * side) < p_habitat).astype(np.uint32)
    if deme.sum() == 0:
        deme[0] = 1
    rng2 = np.random.Generator(np.random.PCG64(turnover_seed))
    turnover = 0.5 + rng2.random(side * side)
    return _base("C4-gaussian-%dx%d" % (side, side), EXPLICIT_GAUSSIAN, width=side, height=side, deme=deme,
                 turnover=turnover, sigma=sigma, nu=nu, seed=seed)


def clustered_habitat(side, frac_habitat=0.6, blur_radius=16.0, noise_seed=3):
    """Thresholded periodic-Gaussian-smoothed white noise: exactly frac_habitat of the cells are habitat."""
    rng = np.random.Generator(np.random.PCG64(noise_seed))
    noise = rng.standard_normal((side, side))
    f = np.fft.fftfreq(side)
    g = np.exp(-2.0 * (math.pi ** 2) * (blur_radius ** 2) * (f[:, None] ** 2 + f[None, :] ** 2))
    smooth = np.fft.ifft2(np.fft.fft2(noise) * g).real
    flat = smooth.ravel()
    n_hab = int(round(frac_habitat * flat.size))
    order = np.argsort(flat, kind="stable")
    hab = np.zeros(flat.size, dtype=bool)
    hab[order[flat.size - n_hab:]] = True
    return hab


def c5_stress(side=4096, deme=4, sigma=5.0, nu=1e-6, sample=0.1, seed=42, noise_seed=3, mask_seed=4, blur_radius=16.0):
    """configs[4]: clustered habitat (60 %), deme 4, rounded Gaussian sigma=5, 10 % of individuals sampled."""
    hab = clustered_habitat(side, 0.6, blur_radius, noise_seed)
    d = hab.astype(np.uint32) * np.uint32(deme)
    n_ind = int(d.sum())
    rng = np.random.Generator(np.random.PCG64(mask_seed))
    mask = (rng.random(n_ind) < sample).astype(np.uint8)
    if mask.sum() == 0:
        mask[0] = 1
    return _base("C5-stress-%dx%d" % (side, side), EXPLICIT_GAUSSIAN, width=side, height=side, deme=d, sigma=sigma,
                 nu=nu, seed=seed, mask=mask)


def c6_bigdeme(width=180, height=64, deme_mean=36_000, sigma=2.0, nu=1e-3, sample=0.01, seed=42, deme_seed=5, mask_seed=6):
    """SURVEY NEXT-4 workload shape: few cells with enormous demes (the paper's fg0size12 map is 180 x 64 cells holding
    4.2e9 individuals; this stand-in keeps the grid and scales the demes so that the sample mask stays
    below 1 GB): log-normal deme sizes, 5 % non-habitat cells, rounded Gaussian dispersal, a thin uniform sample."""
    rng = np.random.Generator(np.random.PCG64(deme_seed))
    n = width * height
    deme = np.maximum(rng.lognormal(mean=math.log(deme_mean) - 0.125, sigma=0.5, size=n), 300.0).astype(np.uint32)
    deme[rng.random(n) < 0.05] = 0
    n_ind = int(deme.astype(np.uint64).sum())
    rng2 = np.random.Generator(np.random.PCG64(mask_seed))
    mask = (rng2.random(n_ind) < sample).astype(np.uint8)
    if mask.sum() == 0:
        mask[0] = 1
    return _base("C6-bigdeme-%dx%d" % (width, height), EXPLICIT_GAUSSIAN, width=width, height=height, deme=deme, sigma=sigma,
                 nu=nu, seed=seed, mask=mask)


def c7_habitat_loss(side=4096, deme=4, sigma=5.0, nu=1e-5, sample=0.1, seed=42, noise_seed=3, mask_seed=7, blur_radius=16.0,
                    frac_now=0.6, frac_past=0.85, switch_k=500):
    """Temporally varying habitat: the C5 landscape after a habitat loss. Today frac_now of the cells
    are habitat (C5's clustered map); before interval switch_k the same smoothed field was thresholded lower, so that frac_past of
    the cells were habitat -- a superset of today's, cell by cell."""
    now = clustered_habitat(side, frac_now, blur_radius, noise_seed)
    past = clustered_habitat(side, frac_past, blur_radius, noise_seed)
    assert not (now & ~past).any()
    d_now = now.astype(np.uint32) * np.uint32(deme)
    d_past = past.astype(np.uint32) * np.uint32(deme)
    rng = np.random.Generator(np.random.PCG64(mask_seed))
    mask = (rng.random(int(d_now.sum())) < sample).astype(np.uint8)
    if mask.sum() == 0:
        mask[0] = 1
    return _base("C7-habitat-loss-%dx%d" % (side, side), EXPLICIT_GAUSSIAN, width=side, height=side, deme=d_now, sigma=sigma, nu=nu,
                 seed=seed, mask=mask, past_deme=d_past[None, :], past_start_k=np.array([switch_k], np.uint32))


def n_individuals(cfg):
    if cfg["kind"] == SPATIALLY_IMPLICIT:
        return int(cfg["local_size"])
    if cfg["deme"] is not None:
        return int(np.asarray(cfg["deme"], dtype=np.uint64).sum())
    return int(cfg["uniform_deme"]) * int(cfg["width"]) * int(cfg["height"])


def n_sampled(cfg):
    return n_individuals(cfg) if cfg["mask"] is None else int(np.count_nonzero(cfg["mask"]))


SCENARIO_KEYS = ("kind", "width", "height", "deme", "uniform_deme", "turnover", "uniform_turnover", "matrix",
                 "sigma", "local_size", "meta_size", "migration", "delta_t", "sampler", "past_deme", "past_start_k")


def scenario_kwargs(cfg):
    return {k: cfg[k] for k in SCENARIO_KEYS}


def full_configs():
    """The five BASELINE.json configs at full size (C3's matrix is 128 MiB, C5's maps ~100 MB)."""
    return [c1_nonspatial(), c2_implicit(), c3_matrix(), c4_gaussian(), c5_stress()]


def small_configs():
    """Reduced versions the oracle finishes in seconds; same structure, several tiles, ragged sizes."""
    return [
        c1_nonspatial(J=3001, nu=2e-3, seed=7),
        c2_implicit(J_local=5003, J_meta=2_000_003, m=0.02, nu=2e-3, seed=8),
        c3_matrix(side=13, deme=7, sigma=1.5, nu=2e-3, seed=9),
        c4_gaussian(side=67, sigma=2.0, nu=1e-3, seed=10),
        c5_stress(side=96, deme=4, sigma=2.5, nu=5e-4, sample=0.3, seed=11, blur_radius=4.0),
    ]
