/*
 * necsim_oracle.c -- CPU ORACLE for the Independent algorithm (TEST INFRASTRUCTURE, not product).
 *
 * Plain, slow, single-threaded C99 restatement of DESIGN.md section 2, which in turn follows
 * /root/reference/PAPER.md (arxiv 2108.05815): section 5.2 (L675-747), 7.1 (L932-967), App. C
 * (L1895-1954), App. G.1 (L2157-2187). Every function cites the passage it follows.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call
 * this. It shares no code, header, table or constant generator with paper_2108_05815_b200/csrc/.
 *
 * Pins (tests/ -m "not gpu"): neglog vs 80-digit ln; event-time search properties and KS/chi^2
 * statistics; Ewens mean and tiny-J closed forms (Eq. B.1);
 * classical coalescence SAD on tiny inputs (App. G.3); alias/gauss table mass checks;
 * invariance to lineage order, partition, epoch length and dedup on/off (L25, L1055).
 * "Parity unpinned": the bit values of the hash RNG (R2: the paper's WyHash/SeaHash
 * mixer is not available; quality is pinned by avalanche/chi^2/correlation tests instead).
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fPIC -shared necsim_oracle.c -o libnecsim_oracle.so -lm
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#include <math.h>

typedef uint32_t u32;
typedef uint64_t u64;
typedef int64_t i64;
typedef unsigned __int128 u128;

/* ------------------------------------------------------------------------------------------- */
/* primeable hash RNG (paper 5.2.1, L693-707: prime() on (seed, location, time))  */
/* ------------------------------------------------------------------------------------------- */
static const u32 MULT[12] = {0x6a09e667u, 0xbb67ae85u, 0x3c6ef373u, 0xa54ff53bu, 0x510e527fu, 0x9b05688du,
                             0x1f83d9abu, 0x5be0cd19u, 0xcbbb9d5du, 0x629a292bu, 0x9159015bu, 0x152fecd9u};
static const u32 KEYC[12] = {0x428a2f98u, 0x71374491u, 0xb5c0fbcfu, 0xe9b5dba5u, 0x3956c25bu, 0x59f111f1u,
                             0x923f82a4u, 0xab1c5ed5u, 0xd807aa98u, 0x12835b01u, 0x243185beu, 0x550c7dc3u};
#define GAMMA 0x6a09e667f3bcc909ull
#define L_SPEC 0xbb67ae8584caa73bull
#define L_DISP 0x3c6ef372fe94f82bull
#define L_INDEX 0xa54ff53a5f1d36f1ull
#define L_MIGR 0x510e527fade682d1ull

/* one Feistel round: p = a*M; (a,b) <- (hi32(p) ^ b ^ K, lo32(p)) */
static void round32(u32 *a, u32 *b, u32 M, u32 K) {
    u64 p = (u64)(*a) * (u64)M;
    u32 na = (u32)(p >> 32) ^ (*b) ^ K;
    *b = (u32)p;
    *a = na;
}

u64 orc_F(u64 x) {
    u32 a = (u32)x, b = (u32)(x >> 32);
    for (int r = 0; r < 6; ++r) round32(&a, &b, MULT[6 + r], KEYC[6 + r]);
    return ((u64)a << 32) | (u64)b;
}

void orc_key_schedule(u64 seed, u32 K[6]) {
    u64 h = orc_F(seed);
    for (int r = 0; r < 6; ++r) K[r] = (u32)(orc_F(h + (u64)(r + 1) * GAMMA) >> 32);
}

u64 orc_prime(const u32 K[6], u32 loc, u32 k) {
    u32 a = loc, b = k;
    for (int r = 0; r < 6; ++r) round32(&a, &b, MULT[r], K[r]);
    return ((u64)a << 32) | (u64)b;
}

static u64 X_of(u64 s, u32 j) { return s + (u64)j * GAMMA; }
u64 orc_draw_time(u64 s, u32 j) { return orc_F(X_of(s, j)); }
u64 orc_draw_spec(u64 s, u32 j) { return orc_F(X_of(s, j) ^ L_SPEC); }
u64 orc_draw_disp(u64 s, u32 j, u32 r) { return orc_F((X_of(s, j) ^ L_DISP) + (u64)r * GAMMA); }
u64 orc_draw_index(u64 s, u32 j) { return orc_F(X_of(s, j) ^ L_INDEX); }
u64 orc_draw_migr(u64 s, u32 j) { return orc_F(X_of(s, j) ^ L_MIGR); }

/* ------------------------------------------------------------------------------------------- */
/* fixed-point -ln (paper Eq. C.3: Exp(lambda) = -log(u)/lambda)           */
/* ------------------------------------------------------------------------------------------- */
typedef struct { u32 Q; u64 A; } neglog_entry;
static const neglog_entry NEGLOG[512] = {
#include "neglog_table.inc"
};
#define LN2_56 49946518145322873ull

u64 orc_neglog(u64 x) {
    u32 z = 0;
    if (x == 0) z = 64; else { u64 v = x; while (!(v >> 63)) { v <<= 1; ++z; } }
    u64 y = (z >= 64) ? 0 : (x << z);
    u64 M = (y >> 14) | 1ull;
    u32 i = (u32)(y >> 54) & 511u;
    u64 P = M * (u64)NEGLOG[i].Q;
    u64 r = P & ((1ull << 61) - 1);
    u32 t = (u32)(r >> 21);
    u32 h1 = 0x55555555u - (t >> 10);
    u32 h2 = 0x80000000u - (u32)((((u64)t * (u64)h1) >> 32) >> 8);
    u64 u = ((u64)t * (u64)h2) >> 32;
    u64 c = ((u64)t * u) >> 24;
    u64 G = NEGLOG[i].A + ((r >> 5) - c);
    u64 Lz = (u64)(z + 1) * LN2_56;
    return Lz > G ? Lz - G : 0;
}

/* scale of 1/mu from binary64 inv = 1/(lambda*delta_t). Returns 0 on success. */
int orc_turnover_scale(double lambda, double delta_t, u32 *Cm, u32 *sh) {
    if (!(lambda > 0.0) || !(delta_t > 0.0) || !isfinite(lambda) || !isfinite(delta_t)) return -1;
    double inv = 1.0 / (lambda * delta_t);
    if (!(inv >= 0x1p-6) || !(inv < 0x1p8)) return -1;
    int ex;
    (void)frexp(inv, &ex);          /* inv = m * 2^ex, m in [0.5,1)  =>  floor(log2 inv) = ex-1 */
    int e = ex - 1;
    double scaled = ldexp(inv, 31 - e); /* exact; in [2^31, 2^32) */
    *Cm = (u32)(u64)floor(scaled);
    *sh = (u32)(7 - e);
    return 0;
}

u64 orc_scale(u64 E, u32 Cm, u32 sh) {
    u64 Eh = E >> 32, El = E & 0xFFFFFFFFull;
    return ((Eh * (u64)Cm) + ((El * (u64)Cm) >> 32)) >> sh;
}

/* real time of (k, f) */
double orc_time(u32 k, u64 f, double delta_t) {
    volatile double a = (double)f * 0x1p-48;
    volatile double b = (double)k + a;
    return b * delta_t;
}

/* ------------------------------------------------------------------------------------------- */
/* event-time search (paper 5.2.2-5.2.3, L719-729)                               */
/* ------------------------------------------------------------------------------------------- */
#define TWO48 (1ull << 48)
/* in/out: *k ; in: f_last (signed, -1 = fresh). out: *j, *T, *s. Returns 0, or -2 if k overflows,
 * or 1 if the search reached interval k_stop without finding an event (then *k == k_stop). */
int orc_next_event(const u32 K[6], u32 loc, u32 *k, i64 f_last, u32 Cm, u32 sh, u32 k_stop,
                   u32 *j_out, u64 *T_out, u64 *s_out) {
    for (;;) {
        if (*k == k_stop) return 1;
        u64 s = orc_prime(K, loc, *k);
        u64 T = 0;
        u32 j = 0;
        for (;;) {
            j += 1;
            T += orc_scale(orc_neglog(orc_draw_time(s, j)), Cm, sh);
            if (T >= TWO48) {
                if (*k == 0xFFFFFFFFu) return -2;
                *k += 1; f_last = -1;
                break;
            }
            if ((i64)T > f_last) { *j_out = j; *T_out = T; *s_out = s; return 0; }
        }
    }
}

/* ------------------------------------------------------------------------------------------- */
/* Poisson / order-statistics event-time sampler (paper 5.2.3 L733-741, C.5 L1940-1954) */
/* ------------------------------------------------------------------------------------------- */
#define L_COUNT 0x9b05688c2b3e6c1full /* frac sqrt 13 */
#define L_THIN 0x1f83d9abfb41bd6bull  /* frac sqrt 17 */
#define ORC_NMAX 256
/* PC[n] = min(floor(P(N <= n) * 2^64), 2^64 - 1), N ~ Poisson(mu): pmf recurrence in binary64 (libm exp) */
void orc_poisson_table(double mu, u64 *PC) {
    double p = exp(-mu), cdf = 0.0;
    for (int n = 0; n < ORC_NMAX; ++n) {
        if (n > 0) p = p * mu / (double)n;
        cdf = cdf + p;
        PC[n] = (cdf >= 1.0) ? 0xFFFFFFFFFFFFFFFFull : (u64)ldexp(cdf, 64);   /* cdf < 1: ldexp exact, conversion truncates */
    }
}
/* number of points of the rate-mu_max stream of (loc, k): N = #{n : c >= PC[n]}, c = F(s ^ L_COUNT) */
u32 orc_poisson_count(const u64 *PC, u64 s) {
    u64 c = orc_F(s ^ L_COUNT);
    u32 n = 0;
    for (int i = 0; i < ORC_NMAX; ++i) if (c >= PC[i]) ++n;
    return n;
}
/* thinning threshold of a cell: point i survives iff thin == 2^32-1 or lo32(F(X_i ^ L_THIN)) < thin */
u32 orc_thin_threshold(double mu_cell, double mu_max) {
    if (mu_cell >= mu_max) return 0xFFFFFFFFu;
    double v = floor((mu_cell / mu_max) * 4294967296.0);
    return (v >= 4294967295.0) ? 0xFFFFFFFFu : (u32)v;
}
/* next point of loc's stream strictly after (k, f_last): all N points of an interval are uniform offsets (order
 * statistics of a Poisson process, L735-741); the next event is the surviving point with the smallest (f, i), f > f_last.
 * Same contract as orc_next_event. */
int orc_next_event_poisson(const u32 K[6], const u64 *PC, u32 thin, u32 loc, u32 *k, i64 f_last, u32 k_stop,
                           u32 *j_out, u64 *T_out, u64 *s_out) {
    for (;;) {
        if (*k == k_stop) return 1;
        u64 s = orc_prime(K, loc, *k);
        u32 N = orc_poisson_count(PC, s);
        u32 best_i = 0; u64 best_f = 0;
        for (u32 i = 1; i <= N; ++i) {
            u64 X = s + (u64)i * GAMMA;
            u64 f = orc_F(X) >> 16;                                      /* Q0.48 offset in units of delta_t */
            if (thin != 0xFFFFFFFFu && (u32)orc_F(X ^ L_THIN) >= thin) continue;   /* thinned out (rate lambda_cell < lambda_max) */
            if ((i64)f <= f_last) continue;                              /* strictly later (L729) */
            if (best_i == 0 || f < best_f) { best_i = i; best_f = f; }   /* ties: smallest i */
        }
        if (best_i) { *j_out = best_i; *T_out = best_f; *s_out = s; return 0; }
        if (*k == 0xFFFFFFFFu) return -2;
        *k += 1; f_last = -1;
    }
}

/* ------------------------------------------------------------------------------------------- */
/* dispersal tables                                                             */
/* ------------------------------------------------------------------------------------------- */
/* rounded-normal thresholds (R15; paper L1216 "discretised normal distribution"). TG has 2R entries. */
int orc_gauss_R(double sigma) { return (int)ceil(10.0 * sigma); }
void orc_gauss_table(double sigma, int R, u32 *TG) {
    for (int i = 0; i < 2 * R; ++i) {
        double z = ((double)(i - R) + 0.5) / sigma;
        double phi = 0.5 * erfc(-z * 0.7071067811865476);
        double v = floor(phi * 4294967296.0);
        TG[i] = (v >= 4294967295.0) ? 0xFFFFFFFFu : (u32)v;
    }
}
int orc_gauss_lookup(const u32 *TG, int R, u32 u) {
    int c = 0;
    for (int i = 0; i < 2 * R; ++i) if (u >= TG[i]) ++c;
    return c - R;
}

/* alias table for one row (R18; Walker/Vose alias method with the construction order of DESIGN 2.5).
 * returns 0, or -1 on invalid weights, -3 if a zero-weight column ends self-accepting. */
int orc_alias_row(const double *w, u32 n, u32 *thresh, u32 *alias) {
    double S = 0.0;
    for (u32 c = 0; c < n; ++c) { if (!(w[c] >= 0.0) || !isfinite(w[c])) return -1; S = S + w[c]; }
    if (!(S > 0.0)) return -1;
    double *p = (double *)malloc(sizeof(double) * n);
    u32 *small = (u32 *)malloc(sizeof(u32) * n), *large = (u32 *)malloc(sizeof(u32) * n);
    u32 ns = 0, nl = 0;
    for (u32 c = 0; c < n; ++c) {
        volatile double num = w[c] * (double)n;
        p[c] = num / S;
        if (p[c] < 1.0) small[ns++] = c; else large[nl++] = c;
    }
    while (ns > 0 && nl > 0) {
        u32 s = small[--ns], l = large[--nl];
        double v = floor(p[s] * 4294967296.0);
        thresh[s] = (v >= 4294967295.0) ? 0xFFFFFFFFu : (u32)v;
        alias[s] = l;
        volatile double sum = p[l] + p[s];
        p[l] = sum - 1.0;
        if (p[l] < 1.0) small[ns++] = l; else large[nl++] = l;
    }
    int rc = 0;
    while (nl > 0) { u32 l = large[--nl]; thresh[l] = 0xFFFFFFFFu; alias[l] = l; if (w[l] == 0.0) rc = -3; }
    while (ns > 0) { u32 s = small[--ns]; thresh[s] = 0xFFFFFFFFu; alias[s] = s; if (w[s] == 0.0) rc = -3; }
    free(p); free(small); free(large);
    return rc;
}

/* ------------------------------------------------------------------------------------------- */
/* Scenario (paper 2.4 L284-302; components L763-784)                                            */
/* ------------------------------------------------------------------------------------------- */
enum { ORC_NONSPATIAL = 0, ORC_SPATIALLY_IMPLICIT = 1, ORC_EXPLICIT_MATRIX = 2, ORC_EXPLICIT_GAUSSIAN = 3 };

typedef struct orc_scenario {
    int kind;
    u32 width, height, ncells;
    u32 *deme;    /* [ncells] */
    u32 *prefix;  /* [ncells+1] */
    u32 *Cm, *sh; /* [ncells] */
    u64 n_locations;     /* all indexed locations */
    u64 n_sampleable;    /* domain of the sample mask */
    /* implicit */
    u64 J_local, J_meta; double migration;
    /* matrix */
    u32 *thresh, *alias; /* [ncells*ncells] */
    /* gaussian */
    double sigma; int R; u32 *TG;
    double delta_t;
    int sampler;         /* 0 exponential (2.4), 1 Poisson / order statistics (2.7) */
    u64 *PC; u32 *thin;  /* Poisson: cdf thresholds of mu_max; per-cell thinning threshold */
    /* temporally varying habitat: era e holds for interval indices k in [era_start[e], era_start[e+1]); era 0 = the
     * present. With eras, `deme` / `prefix` are those of the OLDEST (largest) map: indexed locations are canonical on it. */
    u32 n_eras; u32 *era_deme; u32 *era_start; u32 *prefix0; u32 *deme0;
    double mu_max; double *lam; /* lambda per cell (as given) */
} orc_scenario;

static void set_err(char *err, int errlen, const char *msg) { if (err && errlen > 0) { strncpy(err, msg, (size_t)errlen - 1); err[errlen - 1] = 0; } }

void orc_scenario_destroy(orc_scenario *sc) {
    if (!sc) return;
    free(sc->deme); free(sc->prefix); free(sc->Cm); free(sc->sh); free(sc->thresh); free(sc->alias); free(sc->TG); free(sc->PC); free(sc->thin); free(sc->lam);
    free(sc->era_deme); free(sc->era_start); free(sc->prefix0); free(sc->deme0);
    free(sc);
}

/* deme==NULL: uniform_deme everywhere. turnover==NULL: uniform_turnover everywhere.
 * NONSPATIAL: width=height=1, J = deme of the one cell. SPATIALLY_IMPLICIT: two pseudo-cells
 * (local, meta) built from local_size/meta_size; deme/width/height ignored. */
orc_scenario *orc_scenario_create(int kind, u32 width, u32 height, const u32 *deme, u32 uniform_deme,
                                  const double *turnover, double uniform_turnover, const double *matrix,
                                  double sigma, u64 local_size, u64 meta_size, double migration, double delta_t,
                                  char *err, int errlen) {
    orc_scenario *sc = (orc_scenario *)calloc(1, sizeof(orc_scenario));
    sc->kind = kind; sc->delta_t = delta_t; sc->sigma = sigma; sc->migration = migration;
    if (kind == ORC_SPATIALLY_IMPLICIT) {
        if (local_size == 0 || meta_size == 0 || local_size + meta_size >= (1ull << 32) || !(migration >= 0.0 && migration <= 1.0)) {
            set_err(err, errlen, "implicit: bad sizes or migration"); orc_scenario_destroy(sc); return NULL; }
        sc->width = 2; sc->height = 1; sc->ncells = 2;
        sc->J_local = local_size; sc->J_meta = meta_size;
    } else {
        if (width == 0 || height == 0 || (u64)width * height >= (1ull << 32)) { set_err(err, errlen, "bad width/height"); orc_scenario_destroy(sc); return NULL; }
        if (kind == ORC_NONSPATIAL && !(width == 1 && height == 1)) { set_err(err, errlen, "nonspatial needs 1x1"); orc_scenario_destroy(sc); return NULL; }
        sc->width = width; sc->height = height; sc->ncells = width * height;
    }
    u32 n = sc->ncells;
    sc->deme = (u32 *)malloc(sizeof(u32) * n); sc->prefix = (u32 *)malloc(sizeof(u32) * ((size_t)n + 1));
    sc->Cm = (u32 *)malloc(sizeof(u32) * n); sc->sh = (u32 *)malloc(sizeof(u32) * n);
    sc->lam = (double *)calloc(n, sizeof(double));
    u64 tot = 0;
    for (u32 c = 0; c < n; ++c) {
        u32 d;
        if (kind == ORC_SPATIALLY_IMPLICIT) d = (u32)(c == 0 ? local_size : meta_size);
        else d = deme ? deme[c] : uniform_deme;
        sc->deme[c] = d; sc->prefix[c] = (u32)tot; tot += d;
        double lam = (turnover && kind != ORC_SPATIALLY_IMPLICIT) ? turnover[c] : uniform_turnover;
        sc->lam[c] = lam;
        if (d > 0 || !turnover) {
            if (orc_turnover_scale(lam, delta_t, &sc->Cm[c], &sc->sh[c]) != 0) { set_err(err, errlen, "turnover*delta_t out of range"); orc_scenario_destroy(sc); return NULL; }
        } else { sc->Cm[c] = 0; sc->sh[c] = 0; }
    }
    if (tot == 0 || tot >= (1ull << 32)) { set_err(err, errlen, "number of indexed locations must be in [1, 2^32)"); orc_scenario_destroy(sc); return NULL; }
    sc->prefix[n] = (u32)tot;
    sc->n_locations = tot;
    sc->n_sampleable = (kind == ORC_SPATIALLY_IMPLICIT) ? local_size : tot;
    if (kind == ORC_EXPLICIT_MATRIX) {
        if (!matrix) { set_err(err, errlen, "matrix missing"); orc_scenario_destroy(sc); return NULL; }
        sc->thresh = (u32 *)malloc(sizeof(u32) * (size_t)n * n); sc->alias = (u32 *)malloc(sizeof(u32) * (size_t)n * n);
        for (u32 row = 0; row < n; ++row) {
            if (sc->deme[row] == 0) { for (u32 c = 0; c < n; ++c) { sc->thresh[(size_t)row * n + c] = 0xFFFFFFFFu; sc->alias[(size_t)row * n + c] = c; } continue; }
            for (u32 c = 0; c < n; ++c) if (sc->deme[c] == 0 && matrix[(size_t)row * n + c] != 0.0) { set_err(err, errlen, "dispersal into non-habitat"); orc_scenario_destroy(sc); return NULL; }
            int rc = orc_alias_row(matrix + (size_t)row * n, n, sc->thresh + (size_t)row * n, sc->alias + (size_t)row * n);
            if (rc != 0) { set_err(err, errlen, "bad dispersal matrix row"); orc_scenario_destroy(sc); return NULL; }
        }
    }
    if (kind == ORC_EXPLICIT_GAUSSIAN) {
        if (!(sigma > 0.0) || !isfinite(sigma)) { set_err(err, errlen, "bad sigma"); orc_scenario_destroy(sc); return NULL; }
        sc->R = orc_gauss_R(sigma);
        if ((u32)sc->R >= width || (u32)sc->R >= height) { set_err(err, errlen, "10*sigma must be < min(width,height)"); orc_scenario_destroy(sc); return NULL; }
        sc->TG = (u32 *)malloc(sizeof(u32) * 2 * (size_t)sc->R);
        orc_gauss_table(sigma, sc->R, sc->TG);
    }
    return sc;
}

u64 orc_scenario_num_individuals(const orc_scenario *sc) { return sc->n_sampleable; }

/* Temporally varying habitat (paper 9.3 L1498: "temporally varying landscapes, which enables simulating gradual habitat loss";
 * DESIGN.md 2.8, reading R24). The scenario's deme map is the present (era 0); past_deme[e-1] is the map of era e >= 1, which holds
 * for interval indices k >= past_start_k[e-1] (strictly increasing, > 0). Habitat is only lost towards the present: every era's map
 * contains the younger one cell by cell (an individual of a younger era has a place in every older one). Indexed locations become
 * canonical on the oldest map; the sample mask stays over the present-day individuals. EXPLICIT_GAUSSIAN only. Call before
 * orc_scenario_set_sampler. Returns 0 or -1. */
int orc_scenario_set_eras(orc_scenario *sc, u32 n_past, const u32 *past_deme, const u32 *past_start_k) {
    if (sc->kind != ORC_EXPLICIT_GAUSSIAN || n_past == 0 || sc->n_eras || sc->PC) return -1;
    u32 n = sc->ncells;
    for (u32 e = 0; e < n_past; ++e) {
        if (past_start_k[e] == 0 || (e > 0 && past_start_k[e] <= past_start_k[e - 1])) return -1;
        const u32 *older = past_deme + (size_t)e * n, *younger = e ? past_deme + (size_t)(e - 1) * n : sc->deme;
        for (u32 c = 0; c < n; ++c) if (older[c] < younger[c]) return -1;
    }
    const u32 *oldest = past_deme + (size_t)(n_past - 1) * n;
    u64 tot = 0;
    for (u32 c = 0; c < n; ++c) tot += oldest[c];
    if (tot >= (1ull << 32)) return -1;
    for (u32 c = 0; c < n; ++c)     /* turnover scale wherever any era has habitat */
        if (oldest[c] > 0 && sc->deme[c] == 0 && orc_turnover_scale(sc->lam[c], sc->delta_t, &sc->Cm[c], &sc->sh[c]) != 0) return -1;
    sc->n_eras = n_past + 1;
    sc->era_deme = (u32 *)malloc(sizeof(u32) * (size_t)sc->n_eras * n);
    sc->era_start = (u32 *)malloc(sizeof(u32) * sc->n_eras);
    memcpy(sc->era_deme, sc->deme, sizeof(u32) * n);
    memcpy(sc->era_deme + n, past_deme, sizeof(u32) * (size_t)n_past * n);
    sc->era_start[0] = 0;
    for (u32 e = 0; e < n_past; ++e) sc->era_start[e + 1] = past_start_k[e];
    sc->deme0 = sc->deme; sc->prefix0 = sc->prefix;
    sc->deme = (u32 *)malloc(sizeof(u32) * n); sc->prefix = (u32 *)malloc(sizeof(u32) * ((size_t)n + 1));
    tot = 0;
    for (u32 c = 0; c < n; ++c) { sc->deme[c] = oldest[c]; sc->prefix[c] = (u32)tot; tot += oldest[c]; }
    sc->prefix[n] = (u32)tot;
    sc->n_locations = tot;           /* n_sampleable stays the present-day population */
    return 0;
}
/* deme map in force during interval k */
static const u32 *deme_at(const orc_scenario *sc, u32 k) {
    if (!sc->n_eras) return sc->deme;
    u32 e = 0;
    while (e + 1 < sc->n_eras && sc->era_start[e + 1] <= k) ++e;
    return sc->era_deme + (size_t)e * sc->ncells;
}
/* chooses the event-time sampler (DESIGN.md 2.4 / 2.7). Results depend on it: same law, different realisation. */
int orc_scenario_set_sampler(orc_scenario *sc, int sampler) {
    if (sampler != 0 && sampler != 1) return -1;
    sc->sampler = sampler;
    if (sampler == 1 && !sc->PC) {
        double mu_max = 0.0;
        for (u32 c = 0; c < sc->ncells; ++c) if (sc->deme[c]) { double mu = sc->lam[c] * sc->delta_t; if (mu > mu_max) mu_max = mu; }
        sc->mu_max = mu_max;
        sc->PC = (u64 *)malloc(sizeof(u64) * ORC_NMAX);
        orc_poisson_table(mu_max, sc->PC);
        sc->thin = (u32 *)malloc(sizeof(u32) * sc->ncells);
        for (u32 c = 0; c < sc->ncells; ++c) sc->thin[c] = sc->deme[c] ? orc_thin_threshold(sc->lam[c] * sc->delta_t, mu_max) : 0u;
    }
    return 0;
}
const u64 *orc_scenario_poisson(const orc_scenario *sc, double *mu_max) { *mu_max = sc->mu_max; return sc->PC; }
u32 orc_scenario_thin(const orc_scenario *sc, u32 cell) { return sc->thin ? sc->thin[cell] : 0xFFFFFFFFu; }
const u32 *orc_scenario_thresh(const orc_scenario *sc) { return sc->thresh; }
const u32 *orc_scenario_alias(const orc_scenario *sc) { return sc->alias; }
const u32 *orc_scenario_gauss(const orc_scenario *sc, int *R) { *R = sc->R; return sc->TG; }
void orc_scenario_cell_scale(const orc_scenario *sc, u32 cell, u32 *Cm, u32 *sh) { *Cm = sc->Cm[cell]; *sh = sc->sh[cell]; }

static u32 cell_of_loc(const orc_scenario *sc, u32 loc) {
    /* largest cell with prefix[cell] <= loc and deme[cell] > 0 */
    u32 lo = 0, hi = sc->ncells; /* invariant: prefix[lo] <= loc < prefix[hi] */
    while (hi - lo > 1) { u32 mid = lo + (hi - lo) / 2; if (sc->prefix[mid] <= loc) lo = mid; else hi = mid; }
    return lo;
}

static u64 mulhi64(u64 x, u64 n) { return (u64)(((u128)x * (u128)n) >> 64); }
static int bern(u64 x, u64 thr) { return (x >> 11) < thr; }
u64 orc_thr(double p) { return (u64)floor(ldexp(p, 53)); }

/* DESIGN.md 2.5 step 2. Returns 0 and the new (loc, cell), or -4 if resampling is exhausted. */
static int disperse(const orc_scenario *sc, u64 thr_m, u64 s, u32 k, u32 j, u32 cell, u32 *loc2, u32 *cell2, u64 *resamples) {
    switch (sc->kind) {
    case ORC_NONSPATIAL:
        *loc2 = (u32)mulhi64(orc_draw_disp(s, j, 0), sc->n_locations); *cell2 = 0; return 0;
    case ORC_SPATIALLY_IMPLICIT:
        if (cell == 0 && !bern(orc_draw_migr(s, j), thr_m)) { *loc2 = (u32)mulhi64(orc_draw_disp(s, j, 0), sc->J_local); *cell2 = 0; }
        else { *loc2 = (u32)(sc->J_local + mulhi64(orc_draw_disp(s, j, 0), sc->J_meta)); *cell2 = 1; }
        return 0;
    case ORC_EXPLICIT_MATRIX: {
        u64 x = orc_draw_disp(s, j, 0);
        u32 n = sc->ncells;
        u32 col = (u32)(((x >> 32) * (u64)n) >> 32);
        u32 c2 = ((u32)x < sc->thresh[(size_t)cell * n + col]) ? col : sc->alias[(size_t)cell * n + col];
        u32 d = sc->deme[c2];
        u32 idx = (d == 1) ? 0 : (u32)mulhi64(orc_draw_index(s, j), d);
        *cell2 = c2; *loc2 = sc->prefix[c2] + idx; return 0; }
    case ORC_EXPLICIT_GAUSSIAN: {
        const u32 *deme_k = deme_at(sc, k);   /* the parent lived in the habitat of the event's time (L774, L1498) */
        u32 x0 = cell % sc->width, y0 = cell / sc->width;
        for (u32 r = 0; r < (1u << 20); ++r) {
            u64 x = orc_draw_disp(s, j, r);
            int dx = orc_gauss_lookup(sc->TG, sc->R, (u32)(x >> 32));
            int dy = orc_gauss_lookup(sc->TG, sc->R, (u32)x);
            i64 xx = ((i64)x0 + dx) % (i64)sc->width;  if (xx < 0) xx += sc->width;
            i64 yy = ((i64)y0 + dy) % (i64)sc->height; if (yy < 0) yy += sc->height;
            u32 c2 = (u32)yy * sc->width + (u32)xx;
            u32 d = deme_k[c2];
            if (d > 0) {
                u32 idx = (d == 1) ? 0 : (u32)mulhi64(orc_draw_index(s, j), d);
                *cell2 = c2; *loc2 = sc->prefix[c2] + idx; return 0;
            }
            *resamples += 1;
        }
        return -4; }
    }
    return -1;
}

/* test hook: one dispersal from (loc) at event (k, j) */
int orc_debug_disperse(const orc_scenario *sc, u64 seed, double migration_unused, u32 loc, u32 k, u32 j, u32 *loc2) {
    (void)migration_unused;
    u32 K[6]; orc_key_schedule(seed, K);
    u32 cell = (sc->kind == ORC_SPATIALLY_IMPLICIT) ? (loc >= sc->J_local) : cell_of_loc(sc, loc);
    u32 c2; u64 rs = 0;
    return disperse(sc, orc_thr(sc->migration), orc_prime(K, loc, k), k, j, cell, loc2, &c2, &rs);
}

/* ------------------------------------------------------------------------------------------- */
/* exact dedup: open-addressing map  event (loc,k,j) -> first lineage that executed it            */
/* (paper 7.1.1 L940-946 allows any dedup that never merges distinct trajectories)               */
/* ------------------------------------------------------------------------------------------- */
typedef struct { u64 a, b; } vkey; /* a = loc | k<<32 ; b = j | (id+1)<<32 ; b==0 empty */
typedef struct { vkey *tab; u64 cap, used; } vmap;
static void vmap_init(vmap *m, u64 cap) { m->cap = cap; m->used = 0; m->tab = (vkey *)calloc(cap, sizeof(vkey)); }
static void vmap_clear(vmap *m) { memset(m->tab, 0, m->cap * sizeof(vkey)); m->used = 0; }
static u64 vhash(u64 a, u32 j) { u64 h = a * 0x9E3779B97F4A7C15ull; h ^= h >> 29; h += (u64)j * 0xD6E8FEB86659FD93ull; h ^= h >> 32; return h; }
static void vmap_grow(vmap *m);
/* returns owner id if present, else inserts (id) and returns 0xFFFFFFFF */
static u32 vmap_visit(vmap *m, u32 loc, u32 k, u32 j, u32 id) {
    if ((m->used + 1) * 10 > m->cap * 7) vmap_grow(m);
    u64 a = (u64)loc | ((u64)k << 32);
    u64 h = vhash(a, j) & (m->cap - 1);
    for (;;) {
        vkey *e = &m->tab[h];
        if (e->b == 0) { e->a = a; e->b = (u64)j | ((u64)(id + 1) << 32); m->used++; return 0xFFFFFFFFu; }
        if (e->a == a && (u32)e->b == j) return (u32)(e->b >> 32) - 1;
        h = (h + 1) & (m->cap - 1);
    }
}
static void vmap_grow(vmap *m) {
    vmap n; vmap_init(&n, m->cap * 2);
    for (u64 i = 0; i < m->cap; ++i) if (m->tab[i].b) {
        u64 h = vhash(m->tab[i].a, (u32)m->tab[i].b) & (n.cap - 1);
        while (n.tab[h].b) h = (h + 1) & (n.cap - 1);
        n.tab[h] = m->tab[i]; n.used++;
    }
    free(m->tab); *m = n;
}

/* ------------------------------------------------------------------------------------------- */
/* The simulation (paper 5.2.4 L743-745; outer loop = Water-Level epochs, App. G.1)    */
/* ------------------------------------------------------------------------------------------- */
typedef struct { u32 loc, k, j, pad; u64 f; } orc_event_key;
typedef struct {
    u64 richness, n_lineages, n_events, n_culled, n_epochs, resample_attempts, n_unfinished;
} orc_stats;

typedef struct { u32 loc, k, j; u64 f; u32 abundance; double time; } orc_event;

static int cmp_event(const void *pa, const void *pb) {
    const orc_event_key *a = (const orc_event_key *)pa, *b = (const orc_event_key *)pb;
    if (a->k != b->k) return a->k < b->k ? -1 : 1;
    if (a->f != b->f) return a->f < b->f ? -1 : 1;
    if (a->loc != b->loc) return a->loc < b->loc ? -1 : 1;
    if (a->j != b->j) return a->j < b->j ? -1 : 1;
    return 0;
}

/* Optional sink for the full event stream (paper 6.2 L813-906: Speciation and Dispersal events): every
 * executed event is appended as (origin loc, k, j, f, parent loc or 0xFFFFFFFF for a speciation). With exact dedup each
 * distinct event appears once; the caller sorts by (k, f, loc, j) -- the paper's stream order (event_time, L903, L966). */
static u32 *g_sink_loc, *g_sink_k, *g_sink_j, *g_sink_loc2; static u64 *g_sink_f; static u64 g_sink_cap, *g_sink_n;
void orc_set_event_sink(u32 *loc, u32 *k, u32 *j, u64 *f, u32 *loc2, u64 cap, u64 *n) {
    g_sink_loc = loc; g_sink_k = k; g_sink_j = j; g_sink_f = f; g_sink_loc2 = loc2; g_sink_cap = cap; g_sink_n = n;
    if (n) *n = 0;
}
static void sink_event(u32 loc, u32 k, u32 j, u64 f, u32 loc2) {
    if (!g_sink_n) return;
    u64 i = (*g_sink_n)++;
    if (i < g_sink_cap) { g_sink_loc[i] = loc; g_sink_k[i] = k; g_sink_j[i] = j; g_sink_f[i] = f; g_sink_loc2[i] = loc2; }
}

/*
 * mask: n_sampleable bytes (NULL = all sampled). dedup: 0 off, 1 exact.
 * epoch_events: 0 = one epoch (horizon = never); else the horizon advances so that about that many
 *   events fall into an epoch and the visited-map is cleared at each horizon (G.1).
 * max_steps: 0 = unlimited; else a lineage stops after that many executed events (then it is
 *   "unfinished": label = 0xFFFFFFFF, counted in stats->n_unfinished).
 * Outputs (caller allocates): labels[n_sampled]; events[n_sampled] (first richness entries valid);
 *   per_lineage (optional, may be NULL): terminal key + steps per lineage (own path only; with dedup
 *   on, the key of a culled lineage is the event where it was culled and steps its executed events).
 * Returns 0 or a negative error.
 */
int orc_simulate(const orc_scenario *sc, u64 seed, double nu, const uint8_t *mask, int dedup, u64 epoch_events,
                 u64 max_steps, u32 *labels, orc_event *events, orc_event_key *per_lineage, u32 *per_lineage_steps,
                 orc_stats *stats) {
    memset(stats, 0, sizeof(*stats));
    if (!(nu >= 0.0 && nu <= 1.0)) return -1;
    u32 K[6]; orc_key_schedule(seed, K);
    u64 thr_nu = orc_thr(nu), thr_m = orc_thr(sc->migration);
    /* lineages in canonical order */
    u64 ns = 0;
    for (u64 i = 0; i < sc->n_sampleable; ++i) if (!mask || mask[i]) ++ns;
    if (ns == 0) return -1;
    if (nu == 0.0 && max_steps == 0) return -1;
    u32 *loc = (u32 *)malloc(sizeof(u32) * ns), *cell = (u32 *)malloc(sizeof(u32) * ns), *kk = (u32 *)malloc(sizeof(u32) * ns);
    i64 *ff = (i64 *)malloc(sizeof(i64) * ns);
    u32 *parent = (u32 *)malloc(sizeof(u32) * ns);     /* 0xFFFFFFFF = none */
    u32 *steps = (u32 *)calloc(ns, sizeof(u32));
    uint8_t *state = (uint8_t *)calloc(ns, 1);          /* 0 active, 1 speciated, 2 culled, 3 step-capped */
    orc_event_key *term = (orc_event_key *)calloc(ns, sizeof(orc_event_key));
    u64 n = 0;
    for (u64 i = 0; i < sc->n_sampleable; ++i) if (!mask || mask[i]) {
        if (sc->n_eras) {   /* i counts the present-day individuals; locations are canonical on the oldest map */
            u32 lo = 0, hi = sc->ncells;
            while (hi - lo > 1) { u32 mid = lo + (hi - lo) / 2; if (sc->prefix0[mid] <= (u32)i) lo = mid; else hi = mid; }
            cell[n] = lo; loc[n] = sc->prefix[lo] + ((u32)i - sc->prefix0[lo]);
        } else {
            loc[n] = (u32)i;
            cell[n] = (sc->kind == ORC_SPATIALLY_IMPLICIT) ? 0 : cell_of_loc(sc, (u32)i);
        }
        if (sc->deme[cell[n]] == 0) { n = 0; break; }
        kk[n] = 0; ff[n] = -1; parent[n] = 0xFFFFFFFFu; ++n;
    }
    int rc = 0;
    if (n != ns) rc = -1;
    vmap vis; vis.tab = NULL;
    if (dedup) vmap_init(&vis, 1u << 16);
    u64 active = ns;
    u32 horizon = 0;
    double mu_max = 0.0;
    for (u32 c = 0; c < sc->ncells; ++c) if (sc->deme[c]) { double mu = ldexp(1.0, 24 + (int)sc->sh[c]) / (double)sc->Cm[c]; if (mu > mu_max) mu_max = mu; }
    while (rc == 0 && active > 0) {
        u32 k_stop;
        if (epoch_events == 0) k_stop = 0xFFFFFFFFu;
        else {
            double span = (double)epoch_events / ((double)active * mu_max);
            u64 sp = span < 1.0 ? 1 : (span > 1e9 ? 1000000000ull : (u64)span);
            u64 h = (u64)horizon + sp; k_stop = h >= 0xFFFFFFFFull ? 0xFFFFFFFFu : (u32)h;
        }
        stats->n_epochs++;
        for (u64 id = 0; id < ns && rc == 0; ++id) {
            if (state[id] != 0) continue;
            for (;;) {
                u32 j; u64 T, s;
                int r = sc->sampler == 1
                    ? orc_next_event_poisson(K, sc->PC, sc->thin[cell[id]], loc[id], &kk[id], ff[id], k_stop, &j, &T, &s)
                    : orc_next_event(K, loc[id], &kk[id], ff[id], sc->Cm[cell[id]], sc->sh[cell[id]], k_stop, &j, &T, &s);
                if (r == 1) { ff[id] = -1; break; }          /* reached the horizon: pause (fresh at k_stop) */
                if (r < 0) { rc = r; break; }
                /* event (loc, k, j) at offset T */
                if (dedup) {
                    u32 owner = vmap_visit(&vis, loc[id], kk[id], j, (u32)id);
                    if (owner != 0xFFFFFFFFu) {               /* another lineage executed this event: coalesced (L271, L687) */
                        parent[id] = owner; state[id] = 2; active--; stats->n_culled++;
                        term[id].loc = loc[id]; term[id].k = kk[id]; term[id].j = j; term[id].f = T;
                        break;
                    }
                }
                ff[id] = (i64)T; steps[id]++; stats->n_events++;
                u32 c = cell[id];
                int meta_or_plain = !(sc->kind == ORC_SPATIALLY_IMPLICIT && c == 0);   /* local community: nu = 0 (L1830) */
                if (meta_or_plain && bern(orc_draw_spec(s, j), thr_nu)) {
                    state[id] = 1; active--;
                    term[id].loc = loc[id]; term[id].k = kk[id]; term[id].j = j; term[id].f = T;
                    sink_event(loc[id], kk[id], j, T, 0xFFFFFFFFu);
                    break;
                }
                u32 l2, c2;
                r = disperse(sc, thr_m, s, kk[id], j, c, &l2, &c2, &stats->resample_attempts);
                if (r != 0) { rc = r; break; }
                sink_event(loc[id], kk[id], j, T, l2);
                loc[id] = l2; cell[id] = c2;
                if (max_steps && steps[id] >= max_steps) {
                    state[id] = 3; active--; stats->n_unfinished++;
                    term[id].loc = l2; term[id].k = kk[id]; term[id].j = j; term[id].f = T;
                    break;
                }
            }
        }
        horizon = k_stop;
        if (dedup && epoch_events) vmap_clear(&vis);
        if (k_stop == 0xFFFFFFFFu && active > 0 && rc == 0) rc = -2;
    }
    if (rc == 0) {
        /* resolve: follow parent links to a lineage that ended by itself (L962-967: duplicates merge) */
        orc_event_key *raw = (orc_event_key *)malloc(sizeof(orc_event_key) * ns);
        u64 nraw = 0;
        for (u64 id = 0; id < ns; ++id) if (state[id] == 1) raw[nraw++] = term[id];
        qsort(raw, nraw, sizeof(orc_event_key), cmp_event);
        u64 nu_ = 0;
        for (u64 i = 0; i < nraw; ++i) if (i == 0 || cmp_event(&raw[i], &raw[nu_ - 1]) != 0) raw[nu_++] = raw[i];
        for (u64 e = 0; e < nu_; ++e) {
            events[e].loc = raw[e].loc; events[e].k = raw[e].k; events[e].j = raw[e].j; events[e].f = raw[e].f;
            events[e].abundance = 0; events[e].time = orc_time(raw[e].k, raw[e].f, sc->delta_t);
        }
        for (u64 id = 0; id < ns; ++id) {
            u64 r = id; while (state[r] == 2) r = parent[r];
            if (state[r] != 1) { labels[id] = 0xFFFFFFFFu; continue; }
            /* binary search the root's event */
            u64 lo = 0, hi = nu_;
            while (hi - lo > 1) { u64 mid = lo + (hi - lo) / 2; if (cmp_event(&raw[mid], &term[r]) <= 0) lo = mid; else hi = mid; }
            labels[id] = (u32)lo; events[lo].abundance++;
        }
        stats->richness = nu_;
        free(raw);
    }
    stats->n_lineages = ns;
    if (per_lineage) for (u64 id = 0; id < ns; ++id) { per_lineage[id] = term[id]; }
    if (per_lineage_steps) for (u64 id = 0; id < ns; ++id) per_lineage_steps[id] = steps[id];
    if (dedup) free(vis.tab);
    free(loc); free(cell); free(kk); free(ff); free(parent); free(steps); free(state); free(term);
    return rc;
}

/* ------------------------------------------------------------------------------------------- */
/* Vectorised wrappers of the primitives above (for the pin tests and the GPU parity tests)      */
/* ------------------------------------------------------------------------------------------- */
/* lane: 0 time, 1 spec, 2 disp (attempt r[i]), 3 index, 4 migr, 5 = the primed state s itself */
void orc_batch_draw(u64 seed, int lane, const u32 *loc, const u32 *k, const u32 *j, const u32 *r, u64 *out, u64 n) {
    u32 K[6]; orc_key_schedule(seed, K);
    for (u64 i = 0; i < n; ++i) {
        u64 s = orc_prime(K, loc[i], k[i]);
        switch (lane) {
        case 0: out[i] = orc_draw_time(s, j[i]); break;
        case 1: out[i] = orc_draw_spec(s, j[i]); break;
        case 2: out[i] = orc_draw_disp(s, j[i], r ? r[i] : 0); break;
        case 3: out[i] = orc_draw_index(s, j[i]); break;
        case 4: out[i] = orc_draw_migr(s, j[i]); break;
        default: out[i] = s; break;
        }
    }
}
void orc_batch_F(const u64 *x, u64 *out, u64 n) { for (u64 i = 0; i < n; ++i) out[i] = orc_F(x[i]); }
void orc_batch_neglog(const u64 *x, u64 *out, u64 n) { for (u64 i = 0; i < n; ++i) out[i] = orc_neglog(x[i]); }
/* rc[i] as orc_next_event (k_stop = none) */
void orc_batch_next_event(u64 seed, const u32 *loc, const u32 *k, const i64 *f_last, const u32 *Cm, const u32 *sh,
                          u32 *k_out, u32 *j_out, u64 *T_out, int *rc, u64 n) {
    u32 K[6]; orc_key_schedule(seed, K);
    for (u64 i = 0; i < n; ++i) {
        u32 kk = k[i]; u64 s;
        rc[i] = orc_next_event(K, loc[i], &kk, f_last[i], Cm[i], sh[i], 0xFFFFFFFFu, &j_out[i], &T_out[i], &s);
        k_out[i] = kk;
    }
}
/* Poisson sampler: rc[i] as orc_next_event_poisson with the scenario's table and the thinning threshold of cell[i] */
void orc_batch_next_event_poisson(const orc_scenario *sc, u64 seed, const u32 *loc, const u32 *cell, const u32 *k, const i64 *f_last,
                                  u32 *k_out, u32 *j_out, u64 *T_out, int *rc, u64 n) {
    u32 K[6]; orc_key_schedule(seed, K);
    for (u64 i = 0; i < n; ++i) {
        u32 kk = k[i]; u64 s;
        rc[i] = orc_next_event_poisson(K, sc->PC, sc->thin[cell[i]], loc[i], &kk, f_last[i], 0xFFFFFFFFu, &j_out[i], &T_out[i], &s);
        k_out[i] = kk;
    }
}
void orc_batch_disperse(const orc_scenario *sc, u64 seed, const u32 *loc, const u32 *k, const u32 *j, u32 *loc_out, int *rc, u64 n) {
    for (u64 i = 0; i < n; ++i) rc[i] = orc_debug_disperse(sc, seed, 0.0, loc[i], k[i], j[i], &loc_out[i]);
}
