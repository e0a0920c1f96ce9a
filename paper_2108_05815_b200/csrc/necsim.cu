// necsim.cu -- host side of libnecsim_b200.so: the C-ABI of include/necsim.h.
// Scenario builder (validation, canonical indexing, alias / rounded-normal / turnover-scale tables,
// DESIGN.md 2.4-2.5), the epoch loop around the persistent simulate kernel (Water-Level horizons,
// PAPER.md App. G.1), and the S6 reduction to species. No torch types, no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <stdlib.h>
#include <string>
#include <new>
#include <vector>
#include <algorithm>

#include "../../include/necsim.h"
#include "device_prims.cuh"
#include "sim_types.cuh"
#include "sim_kernel.cuh"
#include "tail_kernel.cuh"
#include "aux_kernels.cuh"
#include "neglog_tables.inc"

using namespace necsim;

static thread_local std::string g_err;
static int fail(int code, const std::string &msg) { g_err = msg; return code; }
#define CU(call)                                                                                         \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return fail(NECSIM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));           \
    } while (0)

extern "C" const char *necsim_last_error(void) { return g_err.c_str(); }

static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// ---------------------------------------------------------------------------------------------------
// host-side table construction
// ---------------------------------------------------------------------------------------------------
// scale of 1/mu from binary64 inv = 1/(lambda*delta_t): Cm = floor(inv * 2^(31-e)), sh = 7 - e, e = floor(log2 inv)
static bool turnover_scale(double lambda, double delta_t, u32 &Cm, u32 &sh) {
    if (!(lambda > 0.0) || !(delta_t > 0.0) || !std::isfinite(lambda) || !std::isfinite(delta_t)) return false;
    double inv = 1.0 / (lambda * delta_t);
    if (!(inv >= 0x1p-6) || !(inv < 0x1p8)) return false;
    int e = ilogb(inv);
    double scaled = scalbn(inv, 31 - e);   // exact, in [2^31, 2^32)
    Cm = (u32)(u64)scaled;                 // truncation = floor for positive values
    sh = (u32)(7 - e);
    return true;
}

static inline u32 to_thresh32(double p) {
    double v = floor(p * 4294967296.0);
    return (v >= 4294967295.0) ? 0xFFFFFFFFu : (u32)v;
}

// Walker alias table of one row, construction order of DESIGN.md 2.5 step 3. 0 ok, -1 bad weights, -3 dead column
static int alias_row(const double *w, u32 n, uint2 *out, std::vector<double> &p, std::vector<u32> &small, std::vector<u32> &large) {
    double S = 0.0;
    for (u32 c = 0; c < n; ++c) {
        if (!(w[c] >= 0.0) || !std::isfinite(w[c])) return -1;
        S = S + w[c];
    }
    if (!(S > 0.0)) return -1;
    small.clear(); large.clear();
    for (u32 c = 0; c < n; ++c) {
        volatile double num = w[c] * (double)n;
        p[c] = num / S;
        if (p[c] < 1.0) small.push_back(c); else large.push_back(c);
    }
    while (!small.empty() && !large.empty()) {
        u32 s = small.back(); small.pop_back();
        u32 l = large.back(); large.pop_back();
        out[s].x = to_thresh32(p[s]); out[s].y = l;
        volatile double sum = p[l] + p[s];
        p[l] = sum - 1.0;
        if (p[l] < 1.0) small.push_back(l); else large.push_back(l);
    }
    int rc = 0;
    for (u32 l : large) { out[l].x = 0xFFFFFFFFu; out[l].y = l; if (w[l] == 0.0) rc = -3; }
    for (u32 s : small) { out[s].x = 0xFFFFFFFFu; out[s].y = s; if (w[s] == 0.0) rc = -3; }
    return rc;
}

// rounded-normal thresholds TG[i] = min(floor(Phi((i - R + 0.5)/sigma) * 2^32), 2^32 - 1), i in [0, 2R)
static void gauss_table(double sigma, int R, std::vector<u32> &tg) {
    tg.resize(2 * (size_t)R);
    for (int i = 0; i < 2 * R; ++i) {
        double z = ((double)(i - R) + 0.5) / sigma;
        double phi = 0.5 * erfc(-z * 0.7071067811865476);
        tg[i] = to_thresh32(phi);
    }
}

// ---------------------------------------------------------------------------------------------------
// scenario handle
// ---------------------------------------------------------------------------------------------------
struct necsim_scenario {
    ScenarioDev dev;
    double migration;
    double mu_max;            // max lambda*delta_t over habitat cells (epoch-horizon policy)
    u64 n_individuals;
    size_t ws_bytes;
    int sm_count;
    SimCounters *h_ctr;       // pinned read-back buffer
    cudaEvent_t ev[4];
    bool tables_uploaded;
};

struct ScenarioLayout {
    size_t off_hab8, off_deme32, off_prefix, off_pois, off_thin, off_scale, off_alias, off_gauss, off_hab64, off_era_hab8, off_era_deme32, off_prefix0, total;
    u32 n_eras;
    u32 ncells, gauss_len, nbx, compact_deme;
    int R;
    bool uniform_deme, need_deme32, per_cell_turnover, compact;
};

// Temporally varying habitat: the per-cell tables are built for the OLDEST map (locations are canonical on it);
// `eff` is the caller's description with that map as its deme map.
struct EraView {
    necsim_scenario_desc eff;
    u32 n_eras;                       // 0 = static
    const u32 *maps[4];               // maps[0] = the present ... maps[n_eras - 1] = the oldest
    u32 start[4];
    std::vector<u32> present;         // the present map when the caller gave uniform_deme only
};
static int era_view(const necsim_scenario_desc *d, EraView &v) {
    v.eff = *d; v.n_eras = 0;
    for (int e = 0; e < 4; ++e) { v.maps[e] = NULL; v.start[e] = 0xFFFFFFFFu; }
    if (!d->n_past_eras) return NECSIM_OK;
    if (d->kind != NECSIM_EXPLICIT_GAUSSIAN) return fail(NECSIM_ERR_UNSUPPORTED, "temporally varying habitat: EXPLICIT_GAUSSIAN only");
    if (d->n_past_eras > 3 || !d->past_deme || !d->past_start_k) return fail(NECSIM_ERR_INVALID_ARG, "eras: at most 3 past eras, with their maps and start intervals");
    if (d->width == 0 || d->height == 0 || (u64)d->width * d->height >= (1ull << 32)) return fail(NECSIM_ERR_INVALID_ARG, "bad width/height");
    const size_t n = (size_t)d->width * d->height;
    if (d->deme) v.maps[0] = d->deme;
    else { v.present.assign(n, d->uniform_deme); v.maps[0] = v.present.data(); }
    v.start[0] = 0;
    for (u32 e = 1; e <= d->n_past_eras; ++e) {
        v.maps[e] = d->past_deme + (size_t)(e - 1) * n; v.start[e] = d->past_start_k[e - 1];
        if (v.start[e] == 0 || (e > 1 && v.start[e] <= v.start[e - 1])) return fail(NECSIM_ERR_INVALID_ARG, "eras: past_start_k must be > 0 and strictly increasing");
        for (size_t c = 0; c < n; ++c)
            if (v.maps[e][c] < v.maps[e - 1][c]) return fail(NECSIM_ERR_INVALID_ARG, "eras: habitat may only be lost towards the present (an older map must contain the younger one)");
    }
    v.n_eras = d->n_past_eras + 1;
    v.eff.deme = v.maps[v.n_eras - 1]; v.eff.n_past_eras = 0; v.eff.past_deme = NULL; v.eff.past_start_k = NULL;
    return NECSIM_OK;
}

static int scenario_layout_static(const necsim_scenario_desc *d, ScenarioLayout &L, bool allow_compact);
static int scenario_layout(const necsim_scenario_desc *d, ScenarioLayout &L) {
    if (!d) return fail(NECSIM_ERR_INVALID_ARG, "desc is NULL");
    EraView v;
    int rc = era_view(d, v);
    if (rc) return rc;
    rc = scenario_layout_static(&v.eff, L, v.n_eras == 0);
    if (rc || !v.n_eras) return rc;
    size_t off = L.total;
    L.n_eras = v.n_eras;
    L.off_era_hab8 = off; off = align256(off + (size_t)v.n_eras * L.ncells);
    if (L.need_deme32) { L.off_era_deme32 = off; off = align256(off + 4 * (size_t)v.n_eras * L.ncells); }
    L.off_prefix0 = off; off = align256(off + 4 * ((size_t)L.ncells + 1));
    L.total = off;
    return NECSIM_OK;
}
static int scenario_layout_static(const necsim_scenario_desc *d, ScenarioLayout &L, bool allow_compact) {
    if (!d) return fail(NECSIM_ERR_INVALID_ARG, "desc is NULL");
    memset(&L, 0, sizeof(L));
    if (d->kind < 0 || d->kind > 3) return fail(NECSIM_ERR_INVALID_ARG, "unknown scenario kind");
    if (d->sampler > 1) return fail(NECSIM_ERR_INVALID_ARG, "unknown event-time sampler");
    if (!(d->delta_t > 0.0) || !std::isfinite(d->delta_t)) return fail(NECSIM_ERR_INVALID_ARG, "delta_t must be > 0 and finite");
    if (d->kind == NECSIM_SPATIALLY_IMPLICIT) {
        if (d->local_size == 0 || d->meta_size == 0 || d->local_size + d->meta_size >= (1ull << 32) || !(d->migration >= 0.0 && d->migration <= 1.0))
            return fail(NECSIM_ERR_INVALID_ARG, "implicit: bad sizes or migration");
        L.ncells = 2; L.uniform_deme = false; L.off_pois = 0; L.total = d->sampler ? align256(8 * NS_POIS_N) : 256;
        return NECSIM_OK;
    }
    if (d->width == 0 || d->height == 0 || (u64)d->width * d->height >= (1ull << 32)) return fail(NECSIM_ERR_INVALID_ARG, "bad width/height");
    if (d->kind == NECSIM_NONSPATIAL && !(d->width == 1 && d->height == 1)) return fail(NECSIM_ERR_INVALID_ARG, "nonspatial needs 1x1");
    L.ncells = d->width * d->height;
    L.uniform_deme = (d->deme == NULL) || d->kind == NECSIM_NONSPATIAL;
    L.per_cell_turnover = (d->turnover != NULL) && d->kind != NECSIM_NONSPATIAL;
    if (!L.uniform_deme) {
        for (u32 c = 0; c < L.ncells; ++c) if (d->deme[c] >= 255u) { L.need_deme32 = true; break; }
    } else if (d->kind >= NECSIM_EXPLICIT_MATRIX && d->uniform_deme >= 255u) L.need_deme32 = true;
    size_t off = 0;
    if (d->kind >= NECSIM_EXPLICIT_MATRIX) {   // explicit kinds always carry the per-cell tables
        L.off_hab8 = off; off = align256(off + L.ncells);
        if (L.need_deme32) { L.off_deme32 = off; off = align256(off + 4 * (size_t)L.ncells); }
        L.off_prefix = off; off = align256(off + 4 * ((size_t)L.ncells + 1));
    }
    if (L.per_cell_turnover) { L.off_scale = off; off = align256(off + 8 * (size_t)L.ncells); }
    if (d->sampler) {
        L.off_pois = off; off = align256(off + 8 * NS_POIS_N);
        if (L.per_cell_turnover) { L.off_thin = off; off = align256(off + 4 * (size_t)L.ncells); }
    }
    if (d->kind == NECSIM_EXPLICIT_MATRIX) {
        if (!d->dispersal_matrix) return fail(NECSIM_ERR_INVALID_ARG, "matrix missing");
        L.off_alias = off; off = align256(off + 8 * (size_t)L.ncells * L.ncells);
    }
    if (d->kind == NECSIM_EXPLICIT_GAUSSIAN) {
        if (!(d->sigma > 0.0) || !std::isfinite(d->sigma)) return fail(NECSIM_ERR_INVALID_ARG, "bad sigma");
        if (d->width > 65536u || d->height > 65536u) return fail(NECSIM_ERR_UNSUPPORTED, "gaussian dispersal: width and height must be <= 65536");
        L.R = (int)ceil(10.0 * d->sigma);
        if ((u32)L.R >= d->width || (u32)L.R >= d->height) return fail(NECSIM_ERR_INVALID_ARG, "10*sigma must be < min(width,height)");
        u32 len = 2; while (len < 2u * (u32)L.R) len <<= 1;
        if (len > 1024u) return fail(NECSIM_ERR_UNSUPPORTED, "sigma too large: the threshold table must fit 1024 entries");
        L.gauss_len = len;
        L.off_gauss = off; off = align256(off + 4 * (size_t)len);
        // compact habitat table: every habitat cell holds the same number of individuals
        u32 D = 0; bool same = true;
        if (L.uniform_deme) D = d->uniform_deme;
        else for (u32 c = 0; c < L.ncells && same; ++c) if (d->deme[c]) { if (!D) D = d->deme[c]; else same = (d->deme[c] == D); }
        if (same && D && allow_compact) {
            L.compact = true; L.compact_deme = D; L.nbx = (d->width + 31u) / 32u;
            L.off_hab64 = off; off = align256(off + 8 * (size_t)L.nbx * 16u * ((d->height + 15u) / 16u));
        }
    }
    L.total = off ? off : 256;
    return NECSIM_OK;
}

extern "C" int necsim_scenario_workspace_size(const necsim_scenario_desc *desc, size_t *device_bytes) {
    if (!device_bytes) return fail(NECSIM_ERR_INVALID_ARG, "device_bytes is NULL");
    ScenarioLayout L;
    int rc = scenario_layout(desc, L);
    if (rc) return rc;
    *device_bytes = L.total;
    return NECSIM_OK;
}

static int upload_neglog_tables(cudaStream_t st) {
    CU(cudaMemcpyToSymbolAsync(NEGLOG_Q_DEV, NEGLOG_Q_HOST, sizeof(NEGLOG_Q_HOST), 0, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyToSymbolAsync(NEGLOG_A_DEV, NEGLOG_A_HOST, sizeof(NEGLOG_A_HOST), 0, cudaMemcpyHostToDevice, st));
    return NECSIM_OK;
}

// no exception crosses the C ABI: host-side allocations (the ncells^2 alias table of EXPLICIT_MATRIX ...) may throw
#define NS_GUARDED(call, on_fail)                                                                        \
    try { return (call); }                                                                               \
    catch (const std::bad_alloc &) { on_fail; return fail(NECSIM_ERR_CAPACITY, "out of host memory"); }   \
    catch (...) { on_fail; return fail(NECSIM_ERR_INVALID_ARG, "unexpected host exception"); }

static int create_scenario_impl(const necsim_scenario_desc *d, void *d_workspace, size_t bytes, void *cuda_stream, necsim_scenario **out);
extern "C" int necsim_create_scenario(const necsim_scenario_desc *d, void *d_workspace, size_t bytes, void *cuda_stream, necsim_scenario **out) {
    NS_GUARDED(create_scenario_impl(d, d_workspace, bytes, cuda_stream, out), if (out) *out = NULL)
}
static int create_scenario_impl(const necsim_scenario_desc *d_caller, void *d_workspace, size_t bytes, void *cuda_stream, necsim_scenario **out) {
    if (!out) return fail(NECSIM_ERR_INVALID_ARG, "out is NULL");
    *out = NULL;
    ScenarioLayout L;
    int rc = scenario_layout(d_caller, L);
    if (rc) return rc;
    EraView era;
    rc = era_view(d_caller, era);
    if (rc) return rc;
    const necsim_scenario_desc *d = &era.eff;      // with eras: the oldest map is the deme map of every table below
    if (!d_workspace || bytes < L.total) return fail(NECSIM_ERR_WORKSPACE_TOO_SMALL, "scenario workspace too small");
    if (((uintptr_t)d_workspace & 255u) != 0) return fail(NECSIM_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev_id = 0, sm_count = 0;
    CU(cudaGetDevice(&dev_id));
    CU(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev_id));

    ScenarioDev sd;
    memset(&sd, 0, sizeof(sd));
    sd.kind = d->kind; sd.delta_t = d->delta_t; sd.width_shift = 0xFFFFFFFFu;
    uint8_t *base = (uint8_t *)d_workspace;
    double mu_max = 0.0, mu_min = 1e300;
    const u32 n = L.ncells;

    if (d->kind == NECSIM_SPATIALLY_IMPLICIT) {
        sd.width = 2; sd.height = 1; sd.ncells = 2;
        sd.J_local = (u32)d->local_size; sd.J_meta = (u32)d->meta_size;
        sd.n_locations = d->local_size + d->meta_size; sd.n_sampleable = d->local_size;
        if (!turnover_scale(d->uniform_turnover, d->delta_t, sd.Cm_u, sd.sh_u)) return fail(NECSIM_ERR_INVALID_ARG, "turnover*delta_t out of range");
        mu_max = mu_min = d->uniform_turnover * d->delta_t;
    } else {
        sd.width = d->width; sd.height = d->height; sd.ncells = n;
        if ((d->width & (d->width - 1)) == 0) { u32 s = 0; while ((1u << s) < d->width) ++s; sd.width_shift = s; }
        // deme, prefix
        u64 tot = 0;
        std::vector<uint8_t> hab8; std::vector<u32> prefix, deme_full;
        const bool tables = d->kind >= NECSIM_EXPLICIT_MATRIX;
        if (L.uniform_deme) {
            u32 ud = d->kind == NECSIM_NONSPATIAL ? (d->deme ? d->deme[0] : d->uniform_deme) : d->uniform_deme;
            sd.uniform_deme = ud; tot = (u64)ud * n;
            if (tables) {
                hab8.assign(n, (uint8_t)std::min(ud, 255u)); prefix.resize((size_t)n + 1);
                for (u32 c = 0; c <= n; ++c) prefix[c] = (u32)std::min<u64>((u64)ud * c, 0xFFFFFFFFull);
                if (L.need_deme32) deme_full.assign(n, ud);
            }
        } else {
            hab8.resize(n); prefix.resize((size_t)n + 1);
            for (u32 c = 0; c < n; ++c) { prefix[c] = (u32)tot; tot += d->deme[c]; hab8[c] = (uint8_t)std::min(d->deme[c], 255u); }
            prefix[n] = (u32)tot;
            if (L.need_deme32) deme_full.assign(d->deme, d->deme + n);
        }
        if (tot == 0 || tot >= (1ull << 32)) return fail(NECSIM_ERR_INVALID_ARG, "number of indexed locations must be in [1, 2^32)");
        sd.n_locations = tot; sd.n_sampleable = tot;
        // turnover scales
        std::vector<uint2> scale;
        if (L.per_cell_turnover) {
            scale.resize(n);
            for (u32 c = 0; c < n; ++c) {
                u32 dm = L.uniform_deme ? sd.uniform_deme : d->deme[c];
                if (dm > 0) {
                    if (!turnover_scale(d->turnover[c], d->delta_t, scale[c].x, scale[c].y)) return fail(NECSIM_ERR_INVALID_ARG, "turnover*delta_t out of range");
                    mu_max = std::max(mu_max, d->turnover[c] * d->delta_t); mu_min = std::min(mu_min, d->turnover[c] * d->delta_t);
                } else scale[c] = make_uint2(0, 0);
            }
            sd.per_cell_turnover = 1;
        } else {
            if (!turnover_scale(d->uniform_turnover, d->delta_t, sd.Cm_u, sd.sh_u)) return fail(NECSIM_ERR_INVALID_ARG, "turnover*delta_t out of range");
            mu_max = mu_min = d->uniform_turnover * d->delta_t;
        }
        if (tables) {
            CU(cudaMemcpyAsync(base + L.off_hab8, hab8.data(), n, cudaMemcpyHostToDevice, st));
            sd.hab8 = base + L.off_hab8;
            if (L.need_deme32) {
                CU(cudaMemcpyAsync(base + L.off_deme32, deme_full.data(), 4 * (size_t)n, cudaMemcpyHostToDevice, st));
                sd.deme32 = (const u32 *)(base + L.off_deme32);
            }
            CU(cudaMemcpyAsync(base + L.off_prefix, prefix.data(), 4 * ((size_t)n + 1), cudaMemcpyHostToDevice, st));
            sd.prefix = (const u32 *)(base + L.off_prefix);
        }
        if (L.per_cell_turnover) {
            CU(cudaMemcpyAsync(base + L.off_scale, scale.data(), 8 * (size_t)n, cudaMemcpyHostToDevice, st));
            sd.scale = (const uint2 *)(base + L.off_scale);
        }
        if (d->kind == NECSIM_EXPLICIT_MATRIX) {
            std::vector<uint2> tab((size_t)n * n);
            std::vector<double> p(n); std::vector<u32> small, large; small.reserve(n); large.reserve(n);
            for (u32 row = 0; row < n; ++row) {
                u32 dm = L.uniform_deme ? sd.uniform_deme : d->deme[row];
                uint2 *o = tab.data() + (size_t)row * n;
                if (dm == 0) { for (u32 c = 0; c < n; ++c) o[c] = make_uint2(0xFFFFFFFFu, c); continue; }
                const double *w = d->dispersal_matrix + (size_t)row * n;
                if (!L.uniform_deme) for (u32 c = 0; c < n; ++c) if (d->deme[c] == 0 && w[c] != 0.0) return fail(NECSIM_ERR_INVALID_ARG, "dispersal into non-habitat");
                if (L.uniform_deme && sd.uniform_deme == 0) return fail(NECSIM_ERR_INVALID_ARG, "no habitat");
                if (alias_row(w, n, o, p, small, large) != 0) return fail(NECSIM_ERR_INVALID_ARG, "bad dispersal matrix row");
            }
            CU(cudaMemcpyAsync(base + L.off_alias, tab.data(), 8 * (size_t)n * n, cudaMemcpyHostToDevice, st));
            CU(cudaStreamSynchronize(st));   // tab goes out of scope
            sd.alias = (const uint2 *)(base + L.off_alias);
        }
        if (d->kind == NECSIM_EXPLICIT_GAUSSIAN) {
            std::vector<u32> tg;
            gauss_table(d->sigma, L.R, tg);
            tg.resize(L.gauss_len, 0xFFFFFFFFu);
            CU(cudaMemcpyAsync(base + L.off_gauss, tg.data(), 4 * (size_t)L.gauss_len, cudaMemcpyHostToDevice, st));
            CU(cudaStreamSynchronize(st));
            sd.gauss = (const u32 *)(base + L.off_gauss); sd.R = L.R; sd.gauss_len = L.gauss_len;
            if (L.compact) {   // {habitat mask, prefix at the block's first cell} per 32-cell block of a row
                std::vector<uint2> hb((size_t)L.nbx * 16u * ((d->height + 15u) / 16u), make_uint2(0u, 0u));   // tiled, see sim_types.cuh
                for (u32 y = 0; y < d->height; ++y)
                    for (u32 b = 0; b < L.nbx; ++b) {
                        u32 m = 0;
                        for (u32 t = 0; t < 32u && b * 32u + t < d->width; ++t) if (hab8[(size_t)y * d->width + b * 32u + t]) m |= 1u << t;
                        hb[(((size_t)(y >> 4) * L.nbx + b) << 4) | (y & 15u)] = make_uint2(m, prefix[(size_t)y * d->width + b * 32u]);
                    }
                CU(cudaMemcpyAsync(base + L.off_hab64, hb.data(), 8 * hb.size(), cudaMemcpyHostToDevice, st));
                CU(cudaStreamSynchronize(st));
                sd.hab64 = (const uint2 *)(base + L.off_hab64); sd.nbx = L.nbx; sd.compact_deme = L.compact_deme;
            }
        }
    }
    if (era.n_eras) {   // per-era habitat maps (the dispersal test of an event of era e) and the present map's prefix sums (S0)
        std::vector<uint8_t> eh((size_t)era.n_eras * n);
        std::vector<u32> ed, p0((size_t)n + 1);
        if (L.need_deme32) ed.resize((size_t)era.n_eras * n);
        for (u32 e = 0; e < era.n_eras; ++e)
            for (u32 c = 0; c < n; ++c) {
                eh[(size_t)e * n + c] = (uint8_t)std::min(era.maps[e][c], 255u);
                if (L.need_deme32) ed[(size_t)e * n + c] = era.maps[e][c];
            }
        u64 tot0 = 0;
        for (u32 c = 0; c < n; ++c) { p0[c] = (u32)tot0; tot0 += era.maps[0][c]; }
        p0[n] = (u32)tot0;
        if (tot0 == 0) return fail(NECSIM_ERR_INVALID_ARG, "eras: the present-day map has no habitat");
        CU(cudaMemcpyAsync(base + L.off_era_hab8, eh.data(), eh.size(), cudaMemcpyHostToDevice, st));
        if (L.need_deme32) CU(cudaMemcpyAsync(base + L.off_era_deme32, ed.data(), 4 * ed.size(), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(base + L.off_prefix0, p0.data(), 4 * p0.size(), cudaMemcpyHostToDevice, st));
        CU(cudaStreamSynchronize(st));
        sd.n_eras = era.n_eras;
        for (int e = 0; e < 4; ++e) sd.era_start[e] = era.start[e];
        sd.era_hab8 = base + L.off_era_hab8;
        sd.era_deme32 = L.need_deme32 ? (const u32 *)(base + L.off_era_deme32) : NULL;
        sd.prefix0 = (const u32 *)(base + L.off_prefix0);
        sd.n_sampleable = tot0;          // the sample mask ranges over the present-day individuals
    }
    sd.sampler = d->sampler;
    sd.margin = (float)(6.1035156e-05 * (1.0 + 1.0 / mu_min));   // NS_MARGIN * (1 + 1/mu_min)
    if (d->sampler) {   // Poisson sampler tables: cdf thresholds of mu_max; per-cell thinning thresholds
        std::vector<u64> pc(NS_POIS_N);
        double p = exp(-mu_max), cdf = 0.0;
        for (u32 nn = 0; nn < NS_POIS_N; ++nn) {
            if (nn > 0) p = p * mu_max / (double)nn;
            cdf = cdf + p;
            pc[nn] = (cdf >= 1.0) ? 0xFFFFFFFFFFFFFFFFull : (u64)ldexp(cdf, 64);
        }
        CU(cudaMemcpyAsync(base + L.off_pois, pc.data(), 8 * NS_POIS_N, cudaMemcpyHostToDevice, st));
        sd.pois = (const u64 *)(base + L.off_pois);
        if (L.per_cell_turnover) {
            std::vector<u32> thin(n);
            for (u32 c = 0; c < n; ++c) {
                const u32 dm = L.uniform_deme ? sd.uniform_deme : d->deme[c];
                const double mu = d->turnover[c] * d->delta_t;
                if (dm == 0) thin[c] = 0;
                else if (mu >= mu_max) thin[c] = 0xFFFFFFFFu;
                else thin[c] = to_thresh32(mu / mu_max);
            }
            CU(cudaMemcpyAsync(base + L.off_thin, thin.data(), 4 * (size_t)n, cudaMemcpyHostToDevice, st));
            sd.thin = (const u32 *)(base + L.off_thin);
        }
        CU(cudaStreamSynchronize(st));
    }
    rc = upload_neglog_tables(st);
    if (rc) return rc;
    CU(cudaStreamSynchronize(st));

    necsim_scenario *h = new necsim_scenario();
    h->dev = sd; h->mu_max = mu_max; h->migration = (d->kind == NECSIM_SPATIALLY_IMPLICIT) ? d->migration : 0.0; h->n_individuals = sd.n_sampleable; h->ws_bytes = L.total; h->sm_count = sm_count;
    h->h_ctr = NULL; h->tables_uploaded = true;
    for (int i = 0; i < 4; ++i) h->ev[i] = NULL;
    if (cudaHostAlloc((void **)&h->h_ctr, sizeof(SimCounters), cudaHostAllocDefault) != cudaSuccess) { delete h; return fail(NECSIM_ERR_CUDA, "cudaHostAlloc failed"); }
    for (int i = 0; i < 4; ++i)
        if (cudaEventCreate(&h->ev[i]) != cudaSuccess) {   // free what exists: the pinned block and the events made so far
            h->ev[i] = NULL;
            necsim_destroy(h);
            return fail(NECSIM_ERR_CUDA, "cudaEventCreate failed");
        }
    *out = h;
    return NECSIM_OK;
}

extern "C" int necsim_scenario_num_individuals(const necsim_scenario *scn, uint64_t *n_individuals) {
    if (!scn || !n_individuals) return fail(NECSIM_ERR_INVALID_ARG, "NULL argument");
    *n_individuals = scn->n_individuals;
    return NECSIM_OK;
}

extern "C" int necsim_destroy(necsim_scenario *scn) {
    if (!scn) return NECSIM_OK;
    if (scn->h_ctr) cudaFreeHost(scn->h_ctr);
    for (int i = 0; i < 4; ++i) if (scn->ev[i]) cudaEventDestroy(scn->ev[i]);
    delete scn;
    return NECSIM_OK;
}

// ---------------------------------------------------------------------------------------------------
// simulate
// ---------------------------------------------------------------------------------------------------
struct ResolvedParams {
    u32 block_threads, grid_blocks, dedup_log2_slots, tail_threshold, probe_mask, probe_mask_tail;
    bool dedup, record;
    u32 stream_fbytes;
    u64 epoch_events, max_steps, ring_cap, stream_cap;
};

static int resolve_params(const necsim_scenario *scn, const necsim_sim_params *p, ResolvedParams &r) {
    necsim_sim_params z;
    memset(&z, 0, sizeof(z));
    if (!p) p = &z;
    r.block_threads = p->block_threads ? p->block_threads : 256u;
    if (r.block_threads % 32u || r.block_threads > 256u) return fail(NECSIM_ERR_INVALID_ARG, "block_threads must be a multiple of 32 and <= 256");
    r.grid_blocks = p->grid_blocks;
    if (p->dedup > 2) return fail(NECSIM_ERR_INVALID_ARG, "dedup must be 0, 1 or 2");
    r.dedup = p->dedup != 2;
    r.dedup_log2_slots = p->dedup_log2_slots ? p->dedup_log2_slots : 22u;
    if (r.dedup_log2_slots < 4 || r.dedup_log2_slots > 28) return fail(NECSIM_ERR_INVALID_ARG, "dedup_log2_slots must be in [4, 28]");
    r.epoch_events = p->epoch_events ? p->epoch_events : (r.dedup ? (1ull << r.dedup_log2_slots) / 2 : 0);
    r.max_steps = p->max_steps;
    if (r.max_steps > 0xFFFFFFFFull) return fail(NECSIM_ERR_INVALID_ARG, "max_steps must fit 32 bits");
    r.tail_threshold = p->tail_threshold;
    r.record = p->record_events != 0;
    if (p->stream_sort_bytes > 5) return fail(NECSIM_ERR_INVALID_ARG, "stream_sort_bytes must be in [0, 5]");
    r.stream_fbytes = p->stream_sort_bytes;   // 0 = chosen per epoch
    r.ring_cap = r.record ? (p->event_ring_capacity ? p->event_ring_capacity : (1ull << 24)) : 0;
    r.stream_cap = r.record ? (p->event_stream_capacity ? p->event_stream_capacity : (1ull << 26)) : 0;
    if (r.ring_cap >= (1ull << 32)) return fail(NECSIM_ERR_INVALID_ARG, "event_ring_capacity must be < 2^32");
    if (p->dedup_probe > 7) return fail(NECSIM_ERR_INVALID_ARG, "dedup_probe must be in [0, 7]");
    {   // probe period 2^pb: the events whose hash has its top pb bits zero. Default: every 8th event (and every 32nd in the tail launch)
        const u32 pb = p->dedup_probe ? p->dedup_probe - 1u : 3u;
        r.probe_mask = pb ? (~0u << (32u - pb)) : 0u;
        r.probe_mask_tail = p->dedup_probe ? r.probe_mask : (~0u << 27);
    }
    (void)scn;
    return NECSIM_OK;
}

struct SimLayout {
    size_t off_ctr, off_qa, off_qb, off_cache, off_term_loc, off_term_k, off_term_j, off_steps, off_parent, off_ring, off_term_f,
        off_state, off_events, off_labels, off_species, off_perm_a, off_perm_b, off_flag, off_hist, off_chunk, off_mask,
        off_scan, off_rec, off_key_a, off_key_b, off_long, off_st_loc, off_st_k, off_st_j, off_st_l2, off_st_f, total;
    u32 n_chunks, sort_blocks;
};

static void sim_layout(u64 n_individuals, u64 cap, const ResolvedParams &rp, SimLayout &L) {
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align256(off + bytes); return o; };
    L.n_chunks = (u32)((n_individuals + NS_CHUNK - 1) / NS_CHUNK);
    const u64 sort_n = std::max<u64>(cap, rp.ring_cap);      // the sort scratch serves the species sort and the per-epoch stream sort
    L.sort_blocks = (u32)((sort_n + NS_SORT_TILE - 1) / NS_SORT_TILE);
    if (L.sort_blocks == 0) L.sort_blocks = 1;
    L.off_ctr = take(sizeof(SimCounters));
    L.off_qa = take(16 * cap); L.off_qb = take(16 * cap);
    L.off_cache = take(rp.dedup ? (16ull << rp.dedup_log2_slots) : 16);
    L.off_term_loc = take(4 * cap); L.off_term_k = take(4 * cap); L.off_term_j = take(4 * cap); L.off_steps = take(4 * cap);
    L.off_parent = take(4 * cap); L.off_ring = take(4 * cap); L.off_term_f = take(8 * cap); L.off_state = take(cap);
    L.off_events = take(sizeof(necsim_event) * cap); L.off_labels = take(4 * cap); L.off_species = take(4 * cap);
    L.off_perm_a = take(4 * sort_n); L.off_perm_b = take(4 * sort_n); L.off_flag = take(4 * sort_n);
    L.off_hist = take(4 * 256 * (size_t)L.sort_blocks); L.off_chunk = take(4 * ((size_t)L.n_chunks + 1));
    L.off_mask = take(n_individuals);
    L.off_scan = take(4 * ((std::max<size_t>(256 * (size_t)L.sort_blocks, sort_n) + NS_SCAN_TILE - 1) / NS_SCAN_TILE + 1));
    L.off_rec = take(32 * rp.ring_cap); L.off_key_a = take(8 * rp.ring_cap); L.off_key_b = take(8 * rp.ring_cap);
    L.off_long = take(8 * (rp.ring_cap / NS_RUN_INLINE + 1));
    L.off_st_loc = take(4 * rp.stream_cap); L.off_st_k = take(4 * rp.stream_cap); L.off_st_j = take(4 * rp.stream_cap);
    L.off_st_l2 = take(4 * rp.stream_cap); L.off_st_f = take(8 * rp.stream_cap);
    L.total = off;
}

extern "C" int necsim_simulate_workspace_size(const necsim_scenario *scn, uint64_t n_sampled, const necsim_sim_params *params, size_t *device_bytes) {
    if (!scn || !device_bytes) return fail(NECSIM_ERR_INVALID_ARG, "NULL argument");
    if (n_sampled == 0 || n_sampled > scn->n_individuals) return fail(NECSIM_ERR_INVALID_ARG, "n_sampled must be in [1, n_individuals]");
    ResolvedParams rp;
    int rc = resolve_params(scn, params, rp);
    if (rc) return rc;
    SimLayout L;
    sim_layout(scn->n_individuals, n_sampled, rp, L);
    *device_bytes = L.total;
    return NECSIM_OK;
}

typedef void (*EpochKernel)(const ScenarioDev, const SimBuffers, const EpochArgs);
// exclusive scan of n u32 on the stream; `sums` = scratch of n / NS_SCAN_TILE + 1 entries; total -> *d_total (may be NULL)
static u32 scan_u32(u32 *a, u32 n, u32 *sums, u32 *d_total, cudaStream_t st) {   // returns the kernels launched
    if (n <= 65536u) { scan_exclusive_kernel<<<1, 1024, 0, st>>>(a, n, d_total); return 1; }
    const u32 nblk = (n + NS_SCAN_TILE - 1) / NS_SCAN_TILE;
    scan_tile_kernel<<<nblk, 1024, 0, st>>>(a, n, sums);
    scan_exclusive_kernel<<<1, 1024, 0, st>>>(sums, nblk, d_total);
    scan_add_kernel<<<nblk, 1024, 0, st>>>(a, n, sums);
    return 3;
}

template <int KIND, bool PERCELL, int SAMP, bool REC, bool COMPACT>
static EpochKernel pick_kernel5(bool dedup, bool tail) {
    if (tail) return dedup ? (EpochKernel)tail_kernel<KIND, true, PERCELL, SAMP, REC, COMPACT> : (EpochKernel)tail_kernel<KIND, false, PERCELL, SAMP, REC, COMPACT>;
    return dedup ? (EpochKernel)simulate_kernel<KIND, true, PERCELL, SAMP, REC, COMPACT> : (EpochKernel)simulate_kernel<KIND, false, PERCELL, SAMP, REC, COMPACT>;
}
// the compact habitat table exists for EXPLICIT_GAUSSIAN only
template <int KIND, bool PERCELL, int SAMP, bool REC>
static EpochKernel pick_kernel4(bool dedup, bool tail, bool compact) {
    if (KIND == 3 && compact) return pick_kernel5<KIND, PERCELL, SAMP, REC, KIND == 3>(dedup, tail);
    return pick_kernel5<KIND, PERCELL, SAMP, REC, false>(dedup, tail);
}
template <int KIND, bool PERCELL>
static EpochKernel pick_kernel2(int sampler, bool rec, bool dedup, bool tail, bool compact) {
    if (sampler) return rec ? pick_kernel4<KIND, PERCELL, 1, true>(dedup, tail, compact) : pick_kernel4<KIND, PERCELL, 1, false>(dedup, tail, compact);
    return rec ? pick_kernel4<KIND, PERCELL, 0, true>(dedup, tail, compact) : pick_kernel4<KIND, PERCELL, 0, false>(dedup, tail, compact);
}
// per-cell turnover exists for the explicit kinds only
static EpochKernel pick_kernel(int kind, bool percell, int sampler, bool rec, bool dedup, bool tail, bool compact) {
    switch (kind) {
    case 0: return pick_kernel2<0, false>(sampler, rec, dedup, tail, false);
    case 1: return pick_kernel2<1, false>(sampler, rec, dedup, tail, false);
    case 2: return percell ? pick_kernel2<2, true>(sampler, rec, dedup, tail, false) : pick_kernel2<2, false>(sampler, rec, dedup, tail, false);
    default: return percell ? pick_kernel2<3, true>(sampler, rec, dedup, tail, compact) : pick_kernel2<3, false>(sampler, rec, dedup, tail, compact);
    }
}
static int occupancy_for(EpochKernel fn, u32 block) {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, (int)block, 0) != cudaSuccess) return 0;
    return nb;
}

#define NS_MIN_EVENTS_PER_LINEAGE 64.0
static u64 thr53(double p) { return (u64)floor(ldexp(p, 53)); }

static int simulate_impl(necsim_scenario *scn, uint64_t seed, double nu, const uint8_t *d_mask, uint64_t cap, const necsim_sim_params *params,
                         void *d_workspace, size_t bytes, cudaStream_t st, necsim_result *out, const SimLayout &L, const ResolvedParams &rp) {
    const ScenarioDev &sd = scn->dev;
    uint8_t *base = (uint8_t *)d_workspace;
    memset(out, 0, sizeof(*out));
    SimBuffers bf;
    memset(&bf, 0, sizeof(bf));
    bf.ctr = (SimCounters *)(base + L.off_ctr);
    uint4 *qa = (uint4 *)(base + L.off_qa), *qb = (uint4 *)(base + L.off_qb);
    bf.cache = (uint4 *)(base + L.off_cache); bf.cache_mask = rp.dedup ? ((1u << rp.dedup_log2_slots) - 1u) : 0u;
    bf.term_loc = (u32 *)(base + L.off_term_loc); bf.term_k = (u32 *)(base + L.off_term_k); bf.term_j = (u32 *)(base + L.off_term_j);
    bf.steps = (u32 *)(base + L.off_steps); bf.parent = (u32 *)(base + L.off_parent); bf.spec_ring = (u32 *)(base + L.off_ring);
    bf.term_f = (u64 *)(base + L.off_term_f); bf.state = base + L.off_state;
    necsim_event *events = (necsim_event *)(base + L.off_events);
    u32 *labels = (u32 *)(base + L.off_labels), *species_of = (u32 *)(base + L.off_species);
    u32 *perm_a = (u32 *)(base + L.off_perm_a), *perm_b = (u32 *)(base + L.off_perm_b), *flag = (u32 *)(base + L.off_flag);
    uint8_t *digit = (uint8_t *)flag;   // the head flags are written after the sort: the same memory holds a pass's digits
    u32 *hist = (u32 *)(base + L.off_hist), *chunk = (u32 *)(base + L.off_chunk), *scan_tmp = (u32 *)(base + L.off_scan);
    bf.rec = (uint4 *)(base + L.off_rec); bf.rec_key = (u64 *)(base + L.off_key_a); bf.rec_cap = (u32)rp.ring_cap;
    u64 *key_a = (u64 *)(base + L.off_key_a), *key_b = (u64 *)(base + L.off_key_b);
    u32 *long_runs = (u32 *)(base + L.off_long);
    const u32 long_cap = (u32)(rp.ring_cap / NS_RUN_INLINE + 1);
    u32 *st_loc = (u32 *)(base + L.off_st_loc), *st_k = (u32 *)(base + L.off_st_k), *st_j = (u32 *)(base + L.off_st_j), *st_l2 = (u32 *)(base + L.off_st_l2);
    u64 *st_f = (u64 *)(base + L.off_st_f);
    u64 stream_n = 0;
    SimCounters *hc = scn->h_ctr;

    if (rp.record) {
        CU(cudaFuncSetAttribute(pair_scatter_kernel<u64, u64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_PAIR_SMEM(8u)));
        CU(cudaFuncSetAttribute(pair_scatter_kernel<u32, u32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)NS_PAIR_SMEM(4u)));
    }
    CU(cudaEventRecord(scn->ev[0], st));
    CU(cudaMemsetAsync(bf.ctr, 0, sizeof(SimCounters), st));
    CU(cudaMemsetAsync(bf.state, 0, cap, st));
    if (rp.dedup) CU(cudaMemsetAsync(bf.cache, 0xFF, 16ull << rp.dedup_log2_slots, st));

    // ---- S0: sample mask -> lineage queue ------------------------------------------------------------
    u64 n_ind = scn->n_individuals;
    u32 n_sampled = 0, n_launch = 0;
    if (d_mask) {
        mask_count_kernel<<<L.n_chunks, 256, 0, st>>>(d_mask, n_ind, chunk);
        scan_exclusive_kernel<<<1, 1024, 0, st>>>(chunk, L.n_chunks, &bf.ctr->n_sampled);
        mask_scatter_kernel<<<L.n_chunks, 256, 0, st>>>(sd, d_mask, n_ind, chunk, qa, (u32)cap);
        n_launch += 3;
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(hc, bf.ctr, sizeof(SimCounters), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        n_sampled = hc->n_sampled;
        if (n_sampled == 0) return fail(NECSIM_ERR_INVALID_ARG, "the sample mask selects nobody");
        if (n_sampled > cap) return fail(NECSIM_ERR_WORKSPACE_TOO_SMALL, "more sampled individuals than n_sampled_capacity");
    } else {
        if (n_ind > cap) return fail(NECSIM_ERR_WORKSPACE_TOO_SMALL, "n_sampled_capacity < n_individuals with a NULL mask");
        n_sampled = (u32)n_ind;
        all_sampled_kernel<<<(n_sampled + 255) / 256, 256, 0, st>>>(sd, n_sampled, qa);
        n_launch += 1;
        CU(cudaGetLastError());
    }

    // ---- S1-S5: epochs of the persistent simulate kernel ---------------------------------------------
    EpochArgs ep;
    ep.key = key_schedule(seed);
    ep.thr_nu = thr53(nu);
    ep.thr_m = thr53(scn->migration);
    ep.max_steps = (u32)rp.max_steps;
    const EpochKernel fn_main = pick_kernel(sd.kind, sd.per_cell_turnover != 0, (int)sd.sampler, rp.record, rp.dedup, false, sd.hab64 != NULL);
    const EpochKernel fn_tail = pick_kernel(sd.kind, sd.per_cell_turnover != 0, (int)sd.sampler, rp.record, rp.dedup, true, sd.hab64 != NULL);
    const int occ = occupancy_for(fn_main, rp.block_threads);
    const int occ_tail = occupancy_for(fn_tail, rp.block_threads);
    ep.probe_mask = rp.probe_mask;
    ep.zero = 0;
    if (occ <= 0 || occ_tail <= 0) return fail(NECSIM_ERR_CUDA, "simulate kernel cannot be resident (occupancy 0)");
    const u32 full_grid = rp.grid_blocks ? rp.grid_blocks : (u32)(occ * scn->sm_count);
    const u32 tail_grid = rp.grid_blocks ? rp.grid_blocks : (u32)(occ_tail * scn->sm_count);
    const u32 warps_per_block = rp.block_threads / 32u;
    // one lineage per warp pays off from about four lineages per resident warp downwards (measured on C5 / C6: sweep in DESIGN.md 5)
    const u32 tail_threshold = rp.tail_threshold ? rp.tail_threshold : 128u * (u32)scn->sm_count;
    const u32 full_cache_mask = rp.dedup ? ((1u << rp.dedup_log2_slots) - 1u) : 0u;
    u32 active = n_sampled, k_start = 0;
    uint4 *q_in = qa, *q_out = qb;
    float ms_sim = 0.f, ms_tail = 0.f;
    u64 n_epochs = 0, n_tail_epochs = 0, ev_before = 0, ev_tail = 0;
    const bool params_default_epoch = !(params && params->epoch_events);
    while (active > 0) {
        u32 k_stop;
        // The tail is ONE launch without a horizon (default policy, no event stream): it is bound by the longest lineage's chain
        // of events, every horizon adds the spread between the slowest and the average lineage of its window, and lineages that
        // have merged keep finding each other through the full-size cache (measured on C5: 5 tail epochs 4.80 s, one 4.24 s, with
        // fewer redundant events).
        const bool unbounded = params_default_epoch && !rp.record && active <= tail_threshold;
        if ((rp.epoch_events == 0 && !rp.record) || unbounded) k_stop = 0xFFFFFFFFu;
        else {
            // (i) tail epochs are latency-bound and their warps stay roughly synchronous in simulated time: longer epochs cost
            // no dedup hits and amortise the end-of-epoch imbalance (spread of events per lineage ~ 1/sqrt(span))
            // (ii) every epoch costs each active lineage a queue round trip and a re-prime, and the kernel a ragged end: by
            // default an epoch holds at least NS_MIN_EVENTS_PER_LINEAGE events per lineage however many lineages there are
            // (measured: 2.9x on the big-deme workload, +5 % redundant events)
            double w = rp.epoch_events ? (double)rp.epoch_events * ((active <= tail_threshold && params_default_epoch) ? 64.0 : 1.0) : 1e30;
            if (params_default_epoch && rp.epoch_events) w = std::max(w, (double)active * NS_MIN_EVENTS_PER_LINEAGE);
            if (rp.record) {   // (iii) the epoch's events (with the redundant ones) must fit the stream ring
                w = std::min(w, 0.5 * (double)rp.ring_cap);
                if ((double)active * scn->mu_max > 0.75 * (double)rp.ring_cap)
                    return fail(NECSIM_ERR_CAPACITY, "event_ring_capacity too small for one interval of the active lineages");
            }
            double span = w / ((double)active * scn->mu_max);
            u64 sp = span < 1.0 ? 1ull : (span > 1e9 ? 1000000000ull : (u64)span);
            if (rp.record) sp = std::min<u64>(sp, (1ull << 24) - 1);   // the record's time key has 24 bits for k - k_start
            u64 h = (u64)k_start + sp;
            k_stop = h >= 0xFFFFFFFFull ? 0xFFFFFFFFu : (u32)h;
        }
        ep.k_start = k_start; ep.k_stop = k_stop;
        const bool tail = active <= tail_threshold;
        // The tail launch probes a subset of the events the per-lane kernel probes (nested masks, so both kernels agree on which of the
        // tail's events probe): with one lineage per warp the exchange sits on the lineage's chain, and a chain of 10^6 events loses
        // nothing by noticing a coalescence 32 instead of 8 events later (C5: 2246 -> 2190 ms per step).
        ep.probe_mask = tail ? rp.probe_mask_tail : rp.probe_mask;
        u32 grid;
        if (tail) {
            ep.lanes_per_warp = 32;
            grid = (u32)std::min<u64>(tail_grid, ((u64)active + warps_per_block - 1) / warps_per_block);
        } else {
            // Fewer lineages than lanes: fill warps, not the machine. A warp's pass costs the same whether 4 or 32 of its lanes hold
            // lineages, and with more than about four warps per scheduler the warps wait for issue slots instead of for their own
            // dependent instructions: 20 000 lineages of C5 spread over all 5 920 resident warps ran at 5.3 us per sequential event,
            // packed into 16 warps per SM at 1.8 us. So: 16 warps per SM (four per scheduler) as full as the lineages make them,
            // more warps only when those are full.
            const u64 total_warps = (u64)full_grid * warps_per_block;
            const u64 few_warps = std::min<u64>(total_warps, 16ull * (u64)scn->sm_count);
            u64 warps = std::min<u64>(total_warps, std::max<u64>(few_warps, ((u64)active + 31) / 32));
            u32 lanes = (u32)std::min<u64>(32, std::max<u64>(1, ((u64)active + warps - 1) / warps));
            ep.lanes_per_warp = lanes;
            grid = (u32)std::min<u64>(full_grid, (warps + warps_per_block - 1) / warps_per_block);
        }
        ep.rec_chunk = 1;
        if (rp.record) {   // chunked ring reservation: at most a quarter (tail) / an eighth (per-lane kernel) of the ring may sit in unused reservations
            const u64 warps = std::max<u64>(1, std::min<u64>(active, (u64)grid * warps_per_block));
            if (tail) ep.rec_chunk = (u32)std::max<u64>(1, std::min<u64>(NS_REC_CHUNK, rp.ring_cap / (4 * warps)));
            else ep.rec_chunk = (u32)std::min<u64>(1024, rp.ring_cap / (8 * warps));      // < 64: the kernel reserves exactly what a pass needs
        }
        bf.q_in = q_in; bf.q_out = q_out; bf.q_in_count = active;
        bf.k_base = rp.record ? k_start : 0u;    // REC kernels: the time key of a record holds k - k_start
        // compact sort keys (see the stream pipeline below): decided before the launch, the kernels write the 32-bit keys themselves
        u32 kbits = 1;
        if (rp.record) { const u64 km = (u64)k_stop - (u64)k_start; while ((1ull << kbits) < km + 1ull) ++kbits; }
        const bool compact_keys = rp.record && !rp.stream_fbytes && kbits <= 16u;
        bf.key_shift = compact_keys ? 8u + kbits : 0u;
        // tail epochs with a horizon: a few thousand synchronous lineages need few slots, keep the footprint (2 MiB) inside L2
        // next to the tables. The tail without a horizon drifts apart in simulated time and needs the long memory of the full cache.
        bf.cache_mask = rp.dedup ? ((tail && !unbounded) ? std::min(full_cache_mask, (1u << 17) - 1u) : full_cache_mask) : 0u;
        CU(cudaMemsetAsync(bf.ctr, 0, 8, st));   // q_head, q_out
        if (rp.record) CU(cudaMemsetAsync(&bf.ctr->n_rec, 0, 4, st));
        CU(cudaEventRecord(scn->ev[2], st));
        (tail ? fn_tail : fn_main)<<<grid, rp.block_threads, 0, st>>>(sd, bf, ep);
        cudaError_t ce = cudaGetLastError();
        if (ce != cudaSuccess) return fail(NECSIM_ERR_CUDA, std::string("simulate kernel launch: ") + cudaGetErrorString(ce));
        CU(cudaEventRecord(scn->ev[3], st));
        CU(cudaMemcpyAsync(hc, bf.ctr, sizeof(SimCounters), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, scn->ev[2], scn->ev[3]));
        ms_sim += ms;
        ++n_epochs; ++n_launch;
        if (getenv("NECSIM_TRACE"))   // per-epoch trace for diagnosis (stderr)
            fprintf(stderr, "[necsim] epoch %llu %s k=[%u,%u) active=%u grid=%u lanes=%u events=%llu culled=%llu ms=%.3f\n", (unsigned long long)n_epochs, tail ? "tail" : "lane",
                    ep.k_start, k_stop, active, grid, ep.lanes_per_warp, (unsigned long long)(hc->n_events - ev_before), (unsigned long long)hc->n_culled, ms);
        if (tail) { ms_tail += ms; ++n_tail_epochs; ev_tail += hc->n_events - ev_before; }
        ev_before = hc->n_events;
        if (hc->error) return fail(NECSIM_ERR_CAPACITY, "interval index overflowed 2^32 or dispersal resampling exhausted");
        if (rp.record && hc->n_rec > 0) {
            // NEXT-3: this epoch's records -> sorted by (k, f, loc, j), duplicates dropped, appended to the stream. Epochs are
            // disjoint windows of simulated time, so the concatenation is globally ordered (Water-Level, G.1 L2157-2187).
            const u32 nr = hc->n_rec;
            if (nr > rp.ring_cap) return fail(NECSIM_ERR_CAPACITY, "event ring overflowed: raise event_ring_capacity");
            const u32 nb = (nr + NS_PAIR_TILE - 1) / NS_PAIR_TILE, g256 = (nr + 255) / 256;
            const u32 kmax = k_stop - ep.k_start;   // (k - k_start) < kmax for every record; the sentinel key ~0 sorts last
            // LSD radix passes over (key, index) pairs. Compact sort (the default when the epoch spans fewer than 2^16 intervals): the
            // interval and the leading bits of f are packed into ONE 32-bit key, ck = key >> (8 + kbits), written by the recording kernels -- 8-byte pairs instead of
            // 12-byte ones, and all 32 - kbits leading bits of f take part (fewer ties than with whole bytes of f). Only the top
            // `passes` bytes of ck are sorted on: the fewest that leave about two records or fewer per prefix value (short runs cost the
            // tie pass less than another radix pass). A forced `stream_sort_bytes` keeps the 64-bit keys (k bytes + that many bytes of f).
            uint8_t *flag8 = (uint8_t *)flag;                                      // (kbits: k - k_start <= kmax - 1 < 2^kbits - 1, all ones = the sentinel only)
            u32 *isrc = NULL, *idst = perm_a, *iother = perm_b;
            CU(cudaMemsetAsync(&bf.ctr->n_long, 0, 4, st));
            if (compact_keys) {
                u32 fbits = 0; while (fbits < 32u - kbits && (double)nr > 2.0 * (double)kmax * (double)(1ull << fbits)) ++fbits;
                const u32 passes = std::min(4u, std::max(1u, (kbits + fbits + 7u) / 8u));
                u32 *k32a = (u32 *)key_b, *k32b = (u32 *)key_b + rp.ring_cap, *ksrc32 = (u32 *)key_a, *kdst32 = k32a;   // the ring's keys are 32-bit already
                for (u32 b = 4u - passes; b < 4u; ++b) {
                    pair_hist_kernel<u32><<<nb, 256, 0, st>>>(ksrc32, nr, 0, 8 * b, hist, nb);
                    n_launch += 2 + scan_u32(hist, 256 * nb, scan_tmp, NULL, st);
                    pair_scatter_kernel<u32, u32><<<nb, NS_PAIR_THREADS, NS_PAIR_SMEM(4u), st>>>(ksrc32, isrc, kdst32, idst, nr, 0, 8 * b, hist, nb);
                    ksrc32 = kdst32; kdst32 = (ksrc32 == k32a) ? k32b : k32a;
                    isrc = idst; std::swap(idst, iother);
                }
                stream_ties_kernel<u32><<<g256, 256, 0, st>>>(ksrc32, isrc, bf.rec, nr, 8 * (4u - passes), flag8, long_runs, &bf.ctr->n_long, long_cap);
            } else {
                // the leading `fbytes` bytes of f (key bytes 5 - fbytes .. 4) and the bytes of k in use (key bytes 5 ..)
                u32 fbytes = rp.stream_fbytes ? std::min(rp.stream_fbytes, 5u) : 1u;
                if (!rp.stream_fbytes)
                    while (fbytes < 5 && (double)nr > 2.0 * (double)kmax * (double)(1ull << (8 * fbytes))) ++fbytes;
                u64 *ksrc = key_a, *kdst = key_b;
                for (u32 b = 5u - fbytes; b < 8; ++b) {
                    if (b >= 5 && (kmax >> (8 * (b - 5))) == 0) continue;
                    pair_hist_kernel<u64><<<nb, 256, 0, st>>>(ksrc, nr, 0, 8 * b, hist, nb);
                    n_launch += 2 + scan_u32(hist, 256 * nb, scan_tmp, NULL, st);
                    pair_scatter_kernel<u64, u64><<<nb, NS_PAIR_THREADS, NS_PAIR_SMEM(8u), st>>>(ksrc, isrc, kdst, idst, nr, 0, 8 * b, hist, nb);
                    std::swap(ksrc, kdst);
                    isrc = idst; std::swap(idst, iother);
                }
                stream_ties_kernel<u64><<<g256, 256, 0, st>>>(ksrc, isrc, bf.rec, nr, 8 * (5u - fbytes), flag8, long_runs, &bf.ctr->n_long, long_cap);
            }
            // isrc: the records' indices sorted by the key prefix; idst: free scratch of the same size
            stream_long_runs_kernel<<<(u32)scn->sm_count * 4u, 256, 0, st>>>(isrc, bf.rec, flag8, long_runs, &bf.ctr->n_long, long_cap, idst);
            const u32 nwt = (nr + NS_WRITE_TILE - 1) / NS_WRITE_TILE;
            u32 *bsum = hist;                                // the histograms are done with: heads per tile of 2048 records
            stream_count_kernel<<<nwt, 256, 0, st>>>(flag8, nr, bsum);
            n_launch += scan_u32(bsum, nwt, scan_tmp, &bf.ctr->q_head, st);   // q_head reused: distinct events of the epoch
            stream_write_kernel<<<nwt, 256, 0, st>>>(bf.rec, isrc, nr, flag8, bsum, stream_n, rp.stream_cap, st_loc, st_k, st_j, st_f, st_l2);
            n_launch += 4;
            CU(cudaGetLastError());
            u32 heads = 0;
            CU(cudaMemcpyAsync(&heads, &bf.ctr->q_head, 4, cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            stream_n += heads;
            if (stream_n > rp.stream_cap) return fail(NECSIM_ERR_CAPACITY, "event stream overflowed: raise event_stream_capacity");
        }
        active = hc->q_out;
        std::swap(q_in, q_out);
        k_start = k_stop;
        if (active > 0 && k_stop == 0xFFFFFFFFu) return fail(NECSIM_ERR_CAPACITY, "lineages still active at interval 2^32-1");
    }
    (void)params; (void)bytes;

    // ---- S6: speciation records -> species (sort / unique / rank), labels, abundances ----------------
    bf.k_base = 0;
    const u32 n_spec = hc->n_spec;
    const u32 j_max = hc->j_max;
    u32 richness = 0;
    if (n_spec > 0) {
        const u32 nb = (n_spec + NS_SORT_TILE - 1) / NS_SORT_TILE;
        const u32 g256 = (n_spec + 255) / 256;
        u32 *src = bf.spec_ring, *dst = perm_a, *other = perm_b;
        // byte b of (j, loc, f, k) is skipped when it is zero for every record
        const u32 maxv[4] = {j_max, (u32)(sd.n_locations - 1), 0, k_start};
        for (u32 b = 0; b < 18; ++b) {
            bool needed;
            if (b < 4) needed = (maxv[0] >> (8 * b)) != 0;
            else if (b < 8) needed = (maxv[1] >> (8 * (b - 4))) != 0;
            else if (b < 14) needed = true;
            else needed = (maxv[3] >> (8 * (b - 14))) != 0;
            if (!needed) continue;
            radix_hist_kernel<<<nb, 256, 0, st>>>(bf, src, n_spec, b, hist, nb, digit);
            n_launch += 2 + scan_u32(hist, 256 * nb, scan_tmp, NULL, st);
            radix_scatter_kernel<<<nb, 256, 0, st>>>(src, dst, n_spec, hist, nb, digit);
            src = dst; std::swap(dst, other);
        }
        CU(cudaGetLastError());
        unique_flag_kernel<<<g256, 256, 0, st>>>(bf, src, n_spec, flag);
        n_launch += scan_u32(flag, n_spec, scan_tmp, &bf.ctr->q_head, st) - 1;   // q_head reused: richness
        unique_write_kernel<<<g256, 256, 0, st>>>(bf, src, n_spec, flag, events, species_of, sd.delta_t);
        n_launch += 3;
        CU(cudaGetLastError());
    }
    // six rounds of pointer jumping bound the walk of label_kernel to 1/64 of the longest chain of links
    if (rp.dedup && hc->n_culled > 0) {
        for (int r = 0; r < 6; ++r) parent_jump_kernel<<<(n_sampled + 255) / 256, 256, 0, st>>>(bf, n_sampled);
        n_launch += 6;
    }
    label_kernel<<<(n_sampled + 255) / 256, 256, 0, st>>>(bf, n_sampled, species_of, events, labels);
    n_launch += 1;
    CU(cudaGetLastError());
    CU(cudaEventRecord(scn->ev[1], st));
    CU(cudaMemcpyAsync(hc, bf.ctr, sizeof(SimCounters), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    richness = n_spec ? hc->q_head : 0;
    float ms_total = 0.f;
    CU(cudaEventElapsedTime(&ms_total, scn->ev[0], scn->ev[1]));

    out->richness = richness; out->n_lineages = n_sampled; out->n_unfinished = hc->n_unfinished;
    out->d_events = events; out->d_labels = labels;
    out->d_term_loc = bf.term_loc; out->d_term_k = bf.term_k; out->d_term_j = bf.term_j; out->d_steps = bf.steps;
    out->d_term_f = bf.term_f; out->d_state = bf.state;
    out->n_events_raw = hc->n_events; out->n_culled = hc->n_culled; out->n_speciation_raw = n_spec; out->n_epochs = n_epochs;
    out->resample_attempts = hc->resamples; out->ms_simulate = ms_sim; out->ms_simulate_tail = ms_tail; out->n_tail_epochs = n_tail_epochs; out->n_events_tail = ev_tail;
    out->ms_total = ms_total; out->n_kernel_launches = n_launch;
    out->n_tail_rounds_exact = hc->tail_rounds_exact;
    if (rp.record) {
        out->d_stream_loc = st_loc; out->d_stream_k = st_k; out->d_stream_j = st_j; out->d_stream_loc2 = st_l2; out->d_stream_f = st_f;
        out->n_stream_events = stream_n;
    }
    return NECSIM_OK;
}

static int simulate_checked(necsim_scenario *scn, uint64_t seed, double nu, const uint8_t *mask, bool mask_on_host, uint64_t cap,
                            const necsim_sim_params *params, void *d_workspace, size_t bytes, void *cuda_stream, necsim_result *out,
                            necsim_event *h_events, uint32_t *h_labels) {
    if (!scn || !out) return fail(NECSIM_ERR_INVALID_ARG, "NULL argument");
    if (!(nu >= 0.0 && nu <= 1.0)) return fail(NECSIM_ERR_INVALID_ARG, "nu must be in [0,1]");
    ResolvedParams rp;
    int rc = resolve_params(scn, params, rp);
    if (rc) return rc;
    if (nu == 0.0 && rp.max_steps == 0) return fail(NECSIM_ERR_INVALID_ARG, "nu = 0 never terminates (set max_steps)");
    if (cap == 0 || cap > scn->n_individuals) return fail(NECSIM_ERR_INVALID_ARG, "n_sampled_capacity must be in [1, n_individuals]");
    SimLayout L;
    sim_layout(scn->n_individuals, cap, rp, L);
    if (!d_workspace || bytes < L.total) return fail(NECSIM_ERR_WORKSPACE_TOO_SMALL, "simulate workspace too small");
    if (((uintptr_t)d_workspace & 255u) != 0) return fail(NECSIM_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint8_t *d_mask = mask;
    if (mask && mask_on_host) {
        uint8_t *stage = (uint8_t *)d_workspace + L.off_mask;
        CU(cudaMemcpyAsync(stage, mask, scn->n_individuals, cudaMemcpyHostToDevice, st));
        d_mask = stage;
    }
    rc = simulate_impl(scn, seed, nu, d_mask, cap, params, d_workspace, bytes, st, out, L, rp);
    if (rc) { cudaStreamSynchronize(st); return rc; }
    if (h_events && out->richness) CU(cudaMemcpyAsync(h_events, out->d_events, sizeof(necsim_event) * out->richness, cudaMemcpyDeviceToHost, st));
    if (h_labels) CU(cudaMemcpyAsync(h_labels, out->d_labels, 4 * out->n_lineages, cudaMemcpyDeviceToHost, st));
    if (h_events || h_labels) CU(cudaStreamSynchronize(st));
    return NECSIM_OK;
}

extern "C" int necsim_simulate(necsim_scenario *scn, uint64_t seed, double nu, const uint8_t *d_sample_mask, uint64_t n_sampled_capacity,
                               const necsim_sim_params *params, void *d_workspace, size_t bytes, void *cuda_stream, necsim_result *out) {
    NS_GUARDED(simulate_checked(scn, seed, nu, d_sample_mask, false, n_sampled_capacity, params, d_workspace, bytes, cuda_stream, out, NULL, NULL), (void)0)
}

extern "C" int necsim_simulate_host(necsim_scenario *scn, uint64_t seed, double nu, const uint8_t *h_sample_mask, uint64_t n_sampled_capacity,
                                    const necsim_sim_params *params, void *d_workspace, size_t bytes, void *cuda_stream, necsim_result *out,
                                    necsim_event *h_events, uint32_t *h_labels) {
    NS_GUARDED(simulate_checked(scn, seed, nu, h_sample_mask, true, n_sampled_capacity, params, d_workspace, bytes, cuda_stream, out, h_events, h_labels), (void)0)
}

// ---------------------------------------------------------------------------------------------------
// merge of species tables (NEXT-2: isolated partitions + merge)
// ---------------------------------------------------------------------------------------------------
struct MergeLayout { size_t off_loc, off_k, off_j, off_f, off_pa, off_pb, off_flag, off_hist, off_cnt, total; u32 nb; };
static void merge_layout(u64 n, MergeLayout &L) {
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align256(off + bytes); return o; };
    L.nb = (u32)((n + NS_SORT_TILE - 1) / NS_SORT_TILE); if (L.nb == 0) L.nb = 1;
    L.off_loc = take(4 * n); L.off_k = take(4 * n); L.off_j = take(4 * n); L.off_f = take(8 * n);
    L.off_pa = take(4 * n); L.off_pb = take(4 * n); L.off_flag = take(4 * n); L.off_hist = take(4 * 256 * (size_t)L.nb); L.off_cnt = take(256);
    L.total = off;
}
extern "C" int necsim_merge_workspace_size(uint64_t n, size_t *device_bytes) {
    if (!device_bytes || n == 0 || n >= (1ull << 32)) return fail(NECSIM_ERR_INVALID_ARG, "n must be in [1, 2^32)");
    MergeLayout L; merge_layout(n, L); *device_bytes = L.total;
    return NECSIM_OK;
}
extern "C" int necsim_merge_species(const necsim_event *d_in, uint64_t n64, void *d_workspace, size_t bytes, void *cuda_stream,
                                    necsim_event *d_out, uint32_t *d_map, uint64_t *richness) {
    if (!d_in || !d_out || !d_map || !richness || n64 == 0 || n64 >= (1ull << 32)) return fail(NECSIM_ERR_INVALID_ARG, "bad argument");
    MergeLayout L; merge_layout(n64, L);
    if (!d_workspace || bytes < L.total) return fail(NECSIM_ERR_WORKSPACE_TOO_SMALL, "merge workspace too small");
    if (((uintptr_t)d_workspace & 255u) != 0) return fail(NECSIM_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const u32 n = (u32)n64, g256 = (n + 255) / 256;
    uint8_t *base = (uint8_t *)d_workspace;
    SimBuffers bf; memset(&bf, 0, sizeof(bf));
    bf.term_loc = (u32 *)(base + L.off_loc); bf.term_k = (u32 *)(base + L.off_k); bf.term_j = (u32 *)(base + L.off_j); bf.term_f = (u64 *)(base + L.off_f);
    u32 *pa = (u32 *)(base + L.off_pa), *pb = (u32 *)(base + L.off_pb), *flag = (u32 *)(base + L.off_flag), *hist = (u32 *)(base + L.off_hist);
    u32 *cnt = (u32 *)(base + L.off_cnt);
    CU(cudaMemsetAsync(d_out, 0, sizeof(necsim_event) * (size_t)n, st));
    merge_unpack_kernel<<<g256, 256, 0, st>>>(d_in, n, bf, pa);
    u32 *src = pa, *dst = pb;
    for (u32 b = 0; b < 18; ++b) {   // all 18 key bytes: the tables are small (thousands of records)
        radix_hist_kernel<<<L.nb, 256, 0, st>>>(bf, src, n, b, hist, L.nb, (uint8_t *)flag);
        scan_exclusive_kernel<<<1, 1024, 0, st>>>(hist, 256 * L.nb, NULL);
        radix_scatter_kernel<<<L.nb, 256, 0, st>>>(src, dst, n, hist, L.nb, (const uint8_t *)flag);
        std::swap(src, dst);
    }
    unique_flag_kernel<<<g256, 256, 0, st>>>(bf, src, n, flag);
    scan_exclusive_kernel<<<1, 1024, 0, st>>>(flag, n, cnt);
    merge_write_kernel<<<g256, 256, 0, st>>>(bf, src, n, flag, d_in, d_out, d_map);
    CU(cudaGetLastError());
    u32 h_cnt = 0;
    CU(cudaMemcpyAsync(&h_cnt, cnt, 4, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    *richness = h_cnt;
    return NECSIM_OK;
}

// ---- the same merge for callers that cannot allocate (CUDA graph capture, serving loops): scratch in a static device array ----------
// The sort / unique scratch of the merge kernels (SoA copy of the records, two permutations, flags, histograms: 32 bytes per record
// and 1 KB per 2048 records) lives in a file-scope __device__ array instead of a caller workspace. Every GPU that loads the library
// holds the array until the process exits. All calls on one device share it: calls that overlap on the GPU (different streams) race.
// Nothing in it has to start at zero -- every kernel of the merge writes what it later reads, for the n of the call -- so the
// previous call's contents do no harm.
#define NS_MERGE_STATIC_BYTES (32u * NECSIM_MERGE_STATIC_MAX + 4u * 256u * (NECSIM_MERGE_STATIC_MAX / NS_SORT_TILE + 1u) + 16u * 256u)
static __device__ __align__(256) unsigned char g_merge_scratch[NS_MERGE_STATIC_BYTES];
#define NS_MAX_DEVICES 64
static void *g_merge_scratch_ptr[NS_MAX_DEVICES];      // device address of g_merge_scratch per device, looked up once with that device current

extern "C" int necsim_merge_species_static(const necsim_event *d_in, uint64_t n64, void *cuda_stream, necsim_event *d_out, uint32_t *d_map,
                                           uint64_t *richness) {
    if (!d_in || !d_out || !d_map || !richness || n64 == 0) return fail(NECSIM_ERR_INVALID_ARG, "bad argument");
    if (n64 > NECSIM_MERGE_STATIC_MAX)
        return fail(NECSIM_ERR_CAPACITY, "necsim_merge_species_static: n exceeds NECSIM_MERGE_STATIC_MAX (65536 records); use necsim_merge_species with a workspace");
    int dev_id = 0;
    CU(cudaGetDevice(&dev_id));
    if (dev_id < 0 || dev_id >= NS_MAX_DEVICES) return fail(NECSIM_ERR_UNSUPPORTED, "device ordinal out of range");
    if (!g_merge_scratch_ptr[dev_id]) {
        // in host code `g_merge_scratch` is only a stand-in for the symbol: its device address comes from the runtime
        void *ptr = NULL;
        CU(cudaGetSymbolAddress(&ptr, g_merge_scratch));
        if (!ptr || ((uintptr_t)ptr & 255u) != 0) return fail(NECSIM_ERR_CUDA, "static merge scratch has no aligned device address");
        g_merge_scratch_ptr[dev_id] = ptr;
    }
    MergeLayout L; merge_layout(n64, L);
    if (L.total > NS_MERGE_STATIC_BYTES) return fail(NECSIM_ERR_CAPACITY, "static merge scratch too small");   // cannot happen for n <= the maximum
    return necsim_merge_species(d_in, n64, g_merge_scratch_ptr[dev_id], NS_MERGE_STATIC_BYTES, cuda_stream, d_out, d_map, richness);
}

// ---------------------------------------------------------------------------------------------------
// test-only exports: device primitives over arrays
// ---------------------------------------------------------------------------------------------------
__global__ void debug_draw_kernel(SeedKey key, int lane_kind, const u32 *loc, const u32 *k, const u32 *j, const u32 *r, u64 *out, u64 n) {
    u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u64 s = prime(key, loc[i], k[i]);
    u64 X = s + (u64)j[i] * NS_GAMMA;
    u64 v;
    switch (lane_kind) {
    case 0: v = draw_time(X); break;
    case 1: v = draw_spec(X); break;
    case 2: v = draw_disp(X, r ? r[i] : 0u); break;
    case 3: v = draw_index(X); break;
    case 4: v = draw_migr(X); break;
    default: v = s; break;
    }
    out[i] = v;
}
__global__ void debug_neglog_kernel(const u64 *x, u64 *out, u64 n) {
    __shared__ unsigned short sQ[512];
    __shared__ u64 sA[512];
    for (u32 i = threadIdx.x; i < 512; i += blockDim.x) { sQ[i] = NEGLOG_Q_DEV[i]; sA[i] = NEGLOG_A_DEV[i]; }
    __syncthreads();
    u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    SmemTables smt; smt.q = smem_addr(sQ); smt.a = smem_addr(sA); smt.tg = smt.g2 = 0;
    if (i < n) out[i] = neglog(x[i], smt);
}
__global__ void debug_next_event_kernel(SeedKey key, const u32 *loc, const u32 *k, const i64 *f_last, const u32 *Cm, const u32 *sh, u32 *k_out,
                                        u32 *j_out, u64 *T_out, int *rc, u64 n) {
    __shared__ unsigned short sQ[512];
    __shared__ u64 sA[512];
    for (u32 i = threadIdx.x; i < 512; i += blockDim.x) { sQ[i] = NEGLOG_Q_DEV[i]; sA[i] = NEGLOG_A_DEV[i]; }
    __syncthreads();
    SmemTables smt; smt.q = smem_addr(sQ); smt.a = smem_addr(sA); smt.tg = smt.g2 = 0;
    u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u32 kk = k[i];
    i64 fl = f_last[i];
    for (;;) {
        u64 X = prime(key, loc[i], kk), T = 0;
        u32 j = 0;
        bool crossed = false;
        for (;;) {
            j += 1; X += NS_GAMMA;
            T += scale_exp(neglog(draw_time(X), smt), Cm[i], sh[i]);
            if (T >= NS_TWO48) { crossed = true; break; }
            if ((i64)T > fl) { k_out[i] = kk; j_out[i] = j; T_out[i] = T; rc[i] = 0; return; }
        }
        if (crossed) {
            if (kk == 0xFFFFFFFFu) { k_out[i] = kk; j_out[i] = 0; T_out[i] = 0; rc[i] = -3; return; }
            kk += 1; fl = -1;
        }
    }
}
template <int KIND>
__global__ void debug_disperse_kernel(const ScenarioDev sc, SeedKey key, u64 thr_m, const u32 *loc, const u32 *k, const u32 *j, u32 *loc_out, u64 n) {
    __shared__ u32 sG[KIND == 3 ? 1024 : 1];
    __shared__ uint2 sG2[KIND == 3 ? NS_G2_LEN : 1];
    if (KIND == 3) gauss_stage(sc, sG, sG2);
    __syncthreads();
    GaussLut gl; gl.tg = smem_addr(sG); gl.g2 = smem_addr(sG2); gl.R = sc.R;
    u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u32 cell = (KIND == 1) ? (loc[i] >= sc.J_local ? 1u : 0u) : cell_of_loc(sc, loc[i]);
    if (KIND == 3) cell = pack_xy(sc, cell);
    u64 X = prime(key, loc[i], k[i]) + (u64)j[i] * NS_GAMMA;
    u32 l2 = 0xFFFFFFFFu, c2 = 0, rs = 0;
    disperse<KIND>(sc, thr_m, X, cell, l2, c2, gl, rs, k[i]);
    loc_out[i] = l2;
}

__global__ void debug_next_event_poisson_kernel(const ScenarioDev sc, SeedKey key, const u32 *loc, const u32 *cell, const u32 *k, const i64 *f_last,
                                                u32 *k_out, u32 *j_out, u64 *T_out, int *rc, u64 n) {
    __shared__ unsigned short sPG[256];
    __shared__ u64 sP[256];
    poisson_stage(sc, sP, sPG);
    SmemTables smt; smt.q = smt.a = smt.tg = smt.g2 = 0; smt.pc = smem_addr(sP); smt.pg = smem_addr(sPG);
    u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const u32 thin = sc.thin ? sc.thin[cell[i]] : 0xFFFFFFFFu;
    u32 kk = k[i];
    i64 fl = f_last[i];
    for (;;) {
        const u64 s = prime(key, loc[i], kk);
        const u32 N = poisson_count(s, smt);
        u32 bi = 0; u64 bf = 0, X = s;
        for (u32 q = 1; q <= N; ++q) {
            X += NS_GAMMA;
            const u64 f = poisson_offset(X);
            if (!poisson_kept(X, thin)) continue;
            if ((i64)f > fl && (bi == 0u || f < bf)) { bi = q; bf = f; }
        }
        if (bi) { k_out[i] = kk; j_out[i] = bi; T_out[i] = bf; rc[i] = 0; return; }
        if (kk == 0xFFFFFFFFu) { k_out[i] = kk; j_out[i] = 0; T_out[i] = 0; rc[i] = -3; return; }
        kk += 1; fl = -1;
    }
}

// the fast round's binary32 offset of one draw beside the exact one, for the error-bound test of the filter
__global__ void debug_approx_time_kernel(const u64 *x, u32 Cm, u32 sh, float *approx, u64 *exact, float *margin, u64 n) {
    __shared__ unsigned short sQ[512];
    __shared__ u64 sA[512];
    for (u32 i = threadIdx.x; i < 512; i += blockDim.x) { sQ[i] = NEGLOG_Q_DEV[i]; sA[i] = NEGLOG_A_DEV[i]; }
    __syncthreads();
    SmemTables smt; smt.q = smem_addr(sQ); smt.a = smem_addr(sA); smt.tg = smt.g2 = 0;
    u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float finv = rate_to_float(Cm, sh);
    approx[i] = approx_exp_time((u32)(x[i] >> 32), NS_LN2F * finv);
    exact[i] = scale_exp(neglog(x[i], smt), Cm, sh);
    if (i == 0) *margin = NS_MARGIN * (1.0f + finv);
}

static inline u32 grid_for(u64 n, u32 block) { return (u32)((n + block - 1) / block); }

extern "C" int necsim_debug_draw(uint64_t seed, int lane, const uint32_t *d_loc, const uint32_t *d_k, const uint32_t *d_j, const uint32_t *d_r,
                                 uint64_t *d_out, uint64_t n, void *cuda_stream) {
    if (n == 0) return NECSIM_OK;
    debug_draw_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)cuda_stream>>>(key_schedule(seed), lane, d_loc, d_k, d_j, d_r, d_out, n);
    CU(cudaGetLastError());
    return NECSIM_OK;
}
extern "C" int necsim_debug_neglog(const uint64_t *d_x, uint64_t *d_out, uint64_t n, void *cuda_stream) {
    if (n == 0) return NECSIM_OK;
    int rc = upload_neglog_tables((cudaStream_t)cuda_stream);
    if (rc) return rc;
    debug_neglog_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)cuda_stream>>>(d_x, d_out, n);
    CU(cudaGetLastError());
    return NECSIM_OK;
}
extern "C" int necsim_debug_approx_time(const uint64_t *d_x, uint32_t Cm, uint32_t sh, float *d_approx, uint64_t *d_exact, float *d_margin, uint64_t n,
                                        void *cuda_stream) {
    if (n == 0) return NECSIM_OK;
    int rc = upload_neglog_tables((cudaStream_t)cuda_stream);
    if (rc) return rc;
    debug_approx_time_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)cuda_stream>>>(d_x, Cm, sh, d_approx, d_exact, d_margin, n);
    CU(cudaGetLastError());
    return NECSIM_OK;
}
extern "C" int necsim_debug_next_event(uint64_t seed, const uint32_t *d_loc, const uint32_t *d_k, const int64_t *d_f_last, const uint32_t *d_Cm,
                                       const uint32_t *d_sh, uint32_t *d_k_out, uint32_t *d_j_out, uint64_t *d_T_out, int32_t *d_rc, uint64_t n,
                                       void *cuda_stream) {
    if (n == 0) return NECSIM_OK;
    int rc = upload_neglog_tables((cudaStream_t)cuda_stream);
    if (rc) return rc;
    debug_next_event_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)cuda_stream>>>(key_schedule(seed), d_loc, d_k, (const i64 *)d_f_last, d_Cm, d_sh,
                                                                                      d_k_out, d_j_out, d_T_out, d_rc, n);
    CU(cudaGetLastError());
    return NECSIM_OK;
}
extern "C" int necsim_debug_disperse(const necsim_scenario *scn, uint64_t seed, const uint32_t *d_loc, const uint32_t *d_k, const uint32_t *d_j,
                                     uint32_t *d_loc_out, uint64_t n, void *cuda_stream) {
    if (!scn) return fail(NECSIM_ERR_INVALID_ARG, "NULL scenario");
    if (n == 0) return NECSIM_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    SeedKey key = key_schedule(seed);
    u64 thr_m = thr53(scn->migration);
    u32 g = grid_for(n, 256);
    switch (scn->dev.kind) {
    case 0: debug_disperse_kernel<0><<<g, 256, 0, st>>>(scn->dev, key, thr_m, d_loc, d_k, d_j, d_loc_out, n); break;
    case 1: debug_disperse_kernel<1><<<g, 256, 0, st>>>(scn->dev, key, thr_m, d_loc, d_k, d_j, d_loc_out, n); break;
    case 2: debug_disperse_kernel<2><<<g, 256, 0, st>>>(scn->dev, key, thr_m, d_loc, d_k, d_j, d_loc_out, n); break;
    default: debug_disperse_kernel<3><<<g, 256, 0, st>>>(scn->dev, key, thr_m, d_loc, d_k, d_j, d_loc_out, n); break;
    }
    CU(cudaGetLastError());
    return NECSIM_OK;
}
extern "C" int necsim_debug_tables(const necsim_scenario *scn, uint32_t *h_thresh, uint32_t *h_alias, uint32_t *h_gauss, int32_t *R_out,
                                   uint32_t *h_Cm, uint32_t *h_sh, void *cuda_stream) {
    if (!scn) return fail(NECSIM_ERR_INVALID_ARG, "NULL scenario");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const ScenarioDev &sd = scn->dev;
    size_t n = sd.ncells;
    if ((h_thresh || h_alias) && sd.alias) {
        std::vector<uint2> tab(n * n);
        CU(cudaMemcpyAsync(tab.data(), sd.alias, 8 * n * n, cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        for (size_t i = 0; i < n * n; ++i) { if (h_thresh) h_thresh[i] = tab[i].x; if (h_alias) h_alias[i] = tab[i].y; }
    }
    if (R_out) *R_out = sd.R;
    if (h_gauss && sd.gauss) {
        CU(cudaMemcpyAsync(h_gauss, sd.gauss, 4 * 2 * (size_t)sd.R, cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    if (h_Cm || h_sh) {
        if (sd.per_cell_turnover) {
            std::vector<uint2> sc(n);
            CU(cudaMemcpyAsync(sc.data(), sd.scale, 8 * n, cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            for (size_t i = 0; i < n; ++i) { if (h_Cm) h_Cm[i] = sc[i].x; if (h_sh) h_sh[i] = sc[i].y; }
        } else {
            for (size_t i = 0; i < n; ++i) { if (h_Cm) h_Cm[i] = sd.Cm_u; if (h_sh) h_sh[i] = sd.sh_u; }
        }
    }
    return NECSIM_OK;
}

extern "C" int necsim_debug_next_event_poisson(const necsim_scenario *scn, uint64_t seed, const uint32_t *d_loc, const uint32_t *d_cell,
                                               const uint32_t *d_k, const int64_t *d_f_last, uint32_t *d_k_out, uint32_t *d_j_out,
                                               uint64_t *d_T_out, int32_t *d_rc, uint64_t n, void *cuda_stream) {
    if (!scn) return fail(NECSIM_ERR_INVALID_ARG, "NULL scenario");
    if (!scn->dev.sampler) return fail(NECSIM_ERR_INVALID_ARG, "the scenario does not use the Poisson sampler");
    if (n == 0) return NECSIM_OK;
    debug_next_event_poisson_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)cuda_stream>>>(scn->dev, key_schedule(seed), d_loc, d_cell, d_k,
                                                                                             (const i64 *)d_f_last, d_k_out, d_j_out, d_T_out, d_rc, n);
    CU(cudaGetLastError());
    return NECSIM_OK;
}
extern "C" int necsim_debug_poisson_table(const necsim_scenario *scn, uint64_t *h_pc, uint32_t *h_thin, double *mu_max, void *cuda_stream) {
    if (!scn) return fail(NECSIM_ERR_INVALID_ARG, "NULL scenario");
    if (!scn->dev.sampler) return fail(NECSIM_ERR_INVALID_ARG, "the scenario does not use the Poisson sampler");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (mu_max) *mu_max = scn->mu_max;
    if (h_pc) CU(cudaMemcpyAsync(h_pc, scn->dev.pois, 8 * NS_POIS_N, cudaMemcpyDeviceToHost, st));
    if (h_thin) {
        if (scn->dev.thin) CU(cudaMemcpyAsync(h_thin, scn->dev.thin, 4 * (size_t)scn->dev.ncells, cudaMemcpyDeviceToHost, st));
        else for (u32 c = 0; c < scn->dev.ncells; ++c) h_thin[c] = 0xFFFFFFFFu;
    }
    CU(cudaStreamSynchronize(st));
    return NECSIM_OK;
}

// ---------------------------------------------------------------------------------------------------
// integer-pipe peak micro-benchmark: independent chains, full occupancy
// ---------------------------------------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(256) int_peak_kernel(u32 iters, u32 *sink) {
    u32 a0 = threadIdx.x * 2654435761u + 1u, a1 = a0 ^ 0x9E3779B9u, a2 = a0 + 0x7F4A7C15u, a3 = a1 * 3u;
    u32 b0 = blockIdx.x + 17u, b1 = b0 ^ 0x85EBCA6Bu, b2 = b0 + 0xC2B2AE35u, b3 = b1 * 5u;
    for (u32 it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (KIND == 0) {   // the hash round: IMAD.WIDE + LOP3 on four independent chains
                feistel(a0, b0, NS_M6, NS_C6); feistel(a1, b1, NS_M7, NS_C7);
                feistel(a2, b2, NS_M8, NS_C8); feistel(a3, b3, NS_M9, NS_C9);
            } else if (KIND == 1) {   // IMAD only
                a0 = a0 * NS_M6 + b0; a1 = a1 * NS_M7 + b1; a2 = a2 * NS_M8 + b2; a3 = a3 * NS_M9 + b3;
                b0 = b0 * NS_M10 + a0; b1 = b1 * NS_M11 + a1; b2 = b2 * NS_M0 + a2; b3 = b3 * NS_M1 + a3;
            } else {   // ALU only: LOP3 / SHF / IADD3
                a0 = (a0 ^ b0 ^ NS_C6) + __funnelshift_l(a0, b0, 7); a1 = (a1 ^ b1 ^ NS_C7) + __funnelshift_l(a1, b1, 9);
                a2 = (a2 ^ b2 ^ NS_C8) + __funnelshift_l(a2, b2, 11); a3 = (a3 ^ b3 ^ NS_C9) + __funnelshift_l(a3, b3, 13);
                b0 = (b0 ^ a0 ^ NS_C10) + __funnelshift_l(b0, a0, 5); b1 = (b1 ^ a1 ^ NS_C11) + __funnelshift_l(b1, a1, 3);
                b2 = (b2 ^ a2 ^ NS_C6) + __funnelshift_l(b2, a2, 15); b3 = (b3 ^ a3 ^ NS_C7) + __funnelshift_l(b3, a3, 17);
            }
        }
    }
    u32 r = a0 ^ a1 ^ a2 ^ a3 ^ b0 ^ b1 ^ b2 ^ b3;
    if (r == 0x12345678u) sink[0] = r;   // keeps the chains alive
}

// random 32-byte-sector gather peak (the denominator for the alias-table and habitat gathers): every thread reads 8 bytes
// from `loads` pseudo-random 32-byte sectors of a table of `sectors` sectors, 8 independent loads in flight
__global__ void __launch_bounds__(256) gather_peak_kernel(const uint2 *table, u64 sectors, u32 loads, u32 *sink) {
    u64 x = ((u64)blockIdx.x * blockDim.x + threadIdx.x) * NS_GAMMA + 0x9E3779B97F4A7C15ull;
    u32 acc = 0;
    for (u32 i = 0; i < loads; i += 8) {
        uint2 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x = x * 6364136223846793005ull + 1442695040888963407ull;
            const u64 sct = __umul64hi(x, sectors);
            asm volatile("ld.global.nc.v2.u32 {%0, %1}, [%2];" : "=r"(v[u].x), "=r"(v[u].y) : "l"(table + 4 * sct));
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) acc ^= v[u].x + v[u].y;
    }
    if (acc == 0x12345678u) sink[0] = acc;
}
extern "C" int necsim_debug_gather_peak(const void *d_table, uint64_t table_bytes, uint32_t loads_per_thread, uint32_t *d_sink, void *cuda_stream,
                                        double *sector_bytes_per_s, float *ms_out) {
    if (!d_table || !d_sink || table_bytes < 32 || loads_per_thread == 0) return fail(NECSIM_ERR_INVALID_ARG, "bad argument");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev_id = 0, sm = 0;
    CU(cudaGetDevice(&dev_id));
    CU(cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev_id));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
    const u32 grid = (u32)sm * 8u, block = 256u, loads = (loads_per_thread + 7u) & ~7u;
    for (int rep = 0; rep < 2; ++rep) {
        if (rep == 1) CU(cudaEventRecord(e0, st));
        gather_peak_kernel<<<grid, block, 0, st>>>((const uint2 *)d_table, table_bytes / 32, loads, d_sink);
    }
    CU(cudaEventRecord(e1, st));
    CU(cudaStreamSynchronize(st));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    if (ms_out) *ms_out = ms;
    if (sector_bytes_per_s) *sector_bytes_per_s = 32.0 * (double)loads * (double)grid * (double)block / ((double)ms * 1e-3);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return NECSIM_OK;
}

extern "C" int necsim_debug_int_peak(int kind, uint32_t iters, uint32_t *d_sink, void *cuda_stream, double *thread_instr_per_s, float *ms_out) {
    if (!d_sink) return fail(NECSIM_ERR_INVALID_ARG, "d_sink is NULL (a 4-byte device buffer of the caller)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev_id = 0, sm = 0;
    CU(cudaGetDevice(&dev_id));
    CU(cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev_id));
    u32 *sink = d_sink;
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
    const u32 grid = (u32)sm * 8u, block = 256u;
    // instructions per inner step: KIND 0: 4 x (IMAD.WIDE + LOP3) = 8; KIND 1: 8 IMAD; KIND 2: 8 x (LOP3 + SHF + IADD3) = 24
    const double per_step = kind == 0 ? 8.0 : (kind == 1 ? 8.0 : 24.0);
    for (int rep = 0; rep < 2; ++rep) {
        if (rep == 1) CU(cudaEventRecord(e0, st));
        if (kind == 0) int_peak_kernel<0><<<grid, block, 0, st>>>(iters, sink);
        else if (kind == 1) int_peak_kernel<1><<<grid, block, 0, st>>>(iters, sink);
        else int_peak_kernel<2><<<grid, block, 0, st>>>(iters, sink);
    }
    CU(cudaEventRecord(e1, st));
    CU(cudaStreamSynchronize(st));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    if (ms_out) *ms_out = ms;
    if (thread_instr_per_s) *thread_instr_per_s = per_step * 8.0 * (double)iters * (double)grid * (double)block / ((double)ms * 1e-3);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return NECSIM_OK;
}
