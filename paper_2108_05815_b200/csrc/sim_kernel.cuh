// sim_kernel.cuh -- the persistent lineage-scheduler kernel.
//
// One lineage per lane (PAPER.md 5.2 L675-747: "each lineage simulated alone"). A lane whose lineage
// ended (speciated / culled as a duplicate / reached the epoch's time horizon / step cap) takes the
// next lineage from the device work queue: one atomicAdd per warp per refill (ballot + popc).
// Every lane is a small state machine: SEARCH (one exponential draw of the event-time search per pass, PAPER.md
// L725-729: sum Exp draws from the interval start until the first partial sum after the lineage's last event) or
// EVENT (duplicate probe + speciation test on the first pass, then one dispersal attempt per pass). Each loop
// iteration the WARP runs the phase that more of its lanes are waiting for (a ballot decides), so both phases
// execute densely instead of the rarer one running at a fraction of the lanes.
#pragma once
#include "sim_types.cuh"

namespace necsim {

#define NS_FULL 0xFFFFFFFFu
#define NS_MAX_RESAMPLE (1u << 20)

__device__ __forceinline__ u32 lanemask_lt() {
    u32 m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// rounded-normal displacement: G(u) = -R + #{i : u >= TG[i]}  (R15). TG is non-decreasing.
// tg: the 2R thresholds in smem. g2: 2048-entry guide indexed by the top 11 bits of u:
//   g2[b].x = pos0 | multi << 16,  pos0 = #{i : TG[i] < b << 21},  g2[b].y = TG[pos0]
//   multi = 1 when bucket b holds two or more thresholds or pos0 == 2R (then the exact forward scan runs).
#define NS_G2_BITS 11
#define NS_G2_LEN (1u << NS_G2_BITS)
struct GaussLut {
    u32 tg, g2;    // shared-window addresses of the thresholds and the guide
    int R;
};
// exact for every u
__device__ __forceinline__ int gauss_disp(const GaussLut &g, u32 u) {
    const uint2 e = lds_v2(g.g2 + 8u * (u >> (32 - NS_G2_BITS)));
    u32 pos = e.x & 0xFFFFu;
    if (e.x >> 16) {
        const u32 n = 2u * (u32)g.R;
        while (pos < n && lds_u32(g.tg + 4u * pos) <= u) ++pos;
    } else {
        pos += (e.y <= u) ? 1u : 0u;
    }
    return (int)pos - g.R;
}
// branch-free variant: `exact` = false where the forward scan would be needed
__device__ __forceinline__ int gauss_disp_fast(const GaussLut &g, u32 u, bool &exact) {
    const uint2 e = lds_v2(g.g2 + 8u * (u >> (32 - NS_G2_BITS)));
    exact = (e.x >> 16) == 0u;
    return (int)((e.x & 0xFFFFu) + ((e.y <= u) ? 1u : 0u)) - g.R;
}
// fills sG / sG2 from the scenario's table (call by all threads of the block; ends with __syncthreads)
__device__ __forceinline__ void gauss_stage(const ScenarioDev &sc, u32 *sG, uint2 *sG2) {
    for (u32 i = threadIdx.x; i < sc.gauss_len; i += blockDim.x) sG[i] = sc.gauss[i];
    __syncthreads();
    const u32 n = 2u * (u32)sc.R;
    for (u32 b = threadIdx.x; b < NS_G2_LEN; b += blockDim.x) {
        // pos0(b) by binary search: first index with TG[i] >= b << 21
        const u32 lim = b << (32 - NS_G2_BITS);
        u32 lo = 0, hi = n;
        while (lo < hi) { u32 mid = (lo + hi) >> 1; if (sG[mid] < lim) lo = mid + 1; else hi = mid; }
        u32 nxt = n;
        if (b + 1 < NS_G2_LEN) {
            const u32 lim2 = (b + 1) << (32 - NS_G2_BITS);
            u32 l2 = lo, h2 = n;
            while (l2 < h2) { u32 mid = (l2 + h2) >> 1; if (sG[mid] < lim2) l2 = mid + 1; else h2 = mid; }
            nxt = l2;
        }
        const u32 multi = (nxt - lo >= 2u || lo == n) ? 1u : 0u;
        sG2[b] = make_uint2(lo | (multi << 16), lo < n ? sG[lo] : 0xFFFFFFFFu);
    }
    __syncthreads();
}

// explicit kinds always have the per-cell tables (hab8 = min(deme, 255), deme32 where needed, prefix)
__device__ __forceinline__ u32 cell_deme(const ScenarioDev &sc, u32 cell) {
    u32 d = __ldg(&sc.hab8[cell]);
    if (d == 255u) d = __ldg(&sc.deme32[cell]);
    return d;
}
__device__ __forceinline__ u32 cell_prefix(const ScenarioDev &sc, u32 cell) { return __ldg(&sc.prefix[cell]); }
// temporally varying habitat: offset of the deme map in force during interval k inside the era tables (0 when static)
__device__ __forceinline__ u32 era_offset(const ScenarioDev &sc, u32 k) {
    if (!sc.n_eras) return 0u;
    const u32 e = (k >= sc.era_start[1] ? 1u : 0u) + (k >= sc.era_start[2] ? 1u : 0u) + (k >= sc.era_start[3] ? 1u : 0u);
    return e * sc.ncells;
}
// deme of a cell at interval k: the static tables, or the era's
__device__ __forceinline__ u32 cell_deme_at(const ScenarioDev &sc, u32 cell, u32 k) {
    if (!sc.n_eras) return cell_deme(sc, cell);
    const u32 o = era_offset(sc, k) + cell;
    u32 d = __ldg(&sc.era_hab8[o]);
    if (d == 255u) d = __ldg(&sc.era_deme32[o]);
    return d;
}

// entry of the compact habitat table that holds cell (xx, yy): the table is tiled, 16 rows of one 32-cell block per 128-byte line
// (sim_types.cuh), so that the targets of one origin's dispersal attempts fall into a handful of lines
__device__ __forceinline__ u32 hab64_index(const ScenarioDev &sc, u32 xx, u32 yy) {
    return ((((yy >> 4) * sc.nbx + (xx >> 5)) << 4) | (yy & 15u));
}
// cell of an indexed location: last cell with prefix[cell] <= loc (that cell has deme > 0)
__device__ __forceinline__ u32 cell_of_loc(const ScenarioDev &sc, u32 loc) {
    if (sc.kind == 0 || sc.kind == 1) return 0;      // non-spatial; implicit: only the local community is sampled
    if (sc.uniform_deme) return loc / sc.uniform_deme;
    u32 lo = 0, hi = sc.ncells;                      // invariant: prefix[lo] <= loc < prefix[hi]
    while (hi - lo > 1) { u32 mid = lo + ((hi - lo) >> 1); if (sc.prefix[mid] <= loc) lo = mid; else hi = mid; }
    return lo;
}
// EXPLICIT_GAUSSIAN lineages carry their cell as packed coordinates (y << 16 | x): no division on the hot path.
__device__ __forceinline__ u32 pack_xy(const ScenarioDev &sc, u32 cell) {
    u32 y = cell / sc.width;
    return (y << 16) | (cell - y * sc.width);
}
__device__ __forceinline__ u32 xy_index(const ScenarioDev &sc, u32 xy) { return (xy >> 16) * sc.width + (xy & 0xFFFFu); }
// torus step of one axis: |d| <= R < size, one wrap suffices (R17)
__device__ __forceinline__ u32 wrap_add(u32 x, int d, u32 size) {
    int v = (int)x + d;
    if (v < 0) v += (int)size; else if (v >= (int)size) v -= (int)size;
    return (u32)v;
}

// DESIGN.md 2.5 step 2: dispersal of the event at stream position X from (loc, cell). Returns false on
// resampling exhaustion. `resamples` counts rejected targets. KIND 3: cell / cell2 are packed (y << 16 | x).
template <int KIND>
__device__ __forceinline__ bool disperse(const ScenarioDev &sc, u64 thr_m, u64 X, u32 cell, u32 &loc2, u32 &cell2,
                                         const GaussLut &gl, u32 &resamples, u32 k = 0) {
    if (KIND == 0) {  // NONSPATIAL: uniform over all J positions, self allowed (R12)
        loc2 = mulhi64_u32(draw_disp(X, 0), (u32)sc.n_locations);
        cell2 = 0;
        return true;
    } else if (KIND == 1) {  // SPATIALLY_IMPLICIT (L294-298, L1830; R13)
        u64 x = draw_disp(X, 0);
        bool to_meta = (cell != 0) || bern(draw_migr(X), thr_m);
        if (to_meta) { loc2 = sc.J_local + mulhi64_u32(x, sc.J_meta); cell2 = 1; }
        else         { loc2 = mulhi64_u32(x, sc.J_local); cell2 = 0; }
        return true;
    } else if (KIND == 2) {  // EXPLICIT_MATRIX: alias-table gather (R18)
        u64 x = draw_disp(X, 0);
        u32 n = sc.ncells;
        u32 col = __umulhi((u32)(x >> 32), n);
        uint2 e = __ldg(&sc.alias[(size_t)cell * n + col]);
        u32 c2 = ((u32)x < e.x) ? col : e.y;
        u32 d = cell_deme(sc, c2);
        u32 idx = (d == 1u) ? 0u : mulhi64_u32(draw_index(X), d);
        cell2 = c2;
        loc2 = cell_prefix(sc, c2) + idx;
        return true;
    } else {  // EXPLICIT_GAUSSIAN: rounded normal on a torus, resample until habitat (R15-R17)
        const u32 x0 = cell & 0xFFFFu, y0 = cell >> 16;
        for (u32 r = 0; r < NS_MAX_RESAMPLE; ++r) {
            const u64 x = draw_disp(X, r);
            const u32 xx = wrap_add(x0, gauss_disp(gl, (u32)(x >> 32)), sc.width);
            const u32 yy = wrap_add(y0, gauss_disp(gl, (u32)x), sc.height);
            const u32 c2 = yy * sc.width + xx;
            const u32 d = cell_deme_at(sc, c2, k);
            if (d > 0) {
                const u32 idx = (d == 1u) ? 0u : mulhi64_u32(draw_index(X), d);
                cell2 = (yy << 16) | xx;
                loc2 = cell_prefix(sc, c2) + idx;
                return true;
            }
            ++resamples;
        }
        return false;
    }
}

// The event's stream position X = prime(loc, k) + j * GAMMA is already a well-mixed function of the event identity (six keyed
// Feistel rounds): folded to 32 bits it chooses the bucket (low bits) and whether the event probes at all (top bits: 3 in the per-lane kernel, 5 in the tail).
// A hit always compares the full key. Every kernel uses this function: entries live across launches.
__device__ __forceinline__ u32 cache_hash(u64 X) { return (u32)X ^ (u32)(X >> 32); }
__device__ __forceinline__ bool cache_probes(u32 h, u32 probe_mask) { return (h & probe_mask) == 0u; }   // probe_mask: the top log2(period) bits

// -ln tables in global memory (filled once per process from neglog_tables.inc), staged to smem per block
__device__ unsigned short NEGLOG_Q_DEV[512];
__device__ u64 NEGLOG_A_DEV[512];

// stages the Poisson cdf thresholds and their top-byte guide (call by all threads of the block; ends with __syncthreads)
__device__ __forceinline__ void poisson_stage(const ScenarioDev &sc, u64 *sP, unsigned short *sPG) {
    for (u32 i = threadIdx.x; i < NS_POIS_N; i += blockDim.x) sP[i] = sc.pois[i];
    __syncthreads();
    for (u32 b = threadIdx.x; b < 256u; b += blockDim.x) {
        const u64 lim = (u64)b << 56;
        u32 n = 0;
        while (n < NS_POIS_N && sP[n] < lim) ++n;
        sPG[b] = (unsigned short)n;
    }
    __syncthreads();
}

// Appends one executed event to the epoch's stream ring (paper 6.2 L813-847: Speciation / Dispersal events).
// Warp-aggregated: the lanes that call this together share one atomicAdd.
#define NS_STREAM_KEY(krel, f) (((u64)(krel) << 40) | ((u64)(f) >> 8))
__device__ __forceinline__ void store_record(const SimBuffers &bf, u32 idx, u32 loc, u32 k, u32 j, u64 f, u32 loc2) {
    // streaming stores (evict first): the ring is written once and read by the sort; it must not push the duplicate-culling cache
    // and the habitat tables out of L2 (measured: L2 hit rate of the recording kernel 41 % with plain stores)
    __stcs(&bf.rec[2u * idx], make_uint4(loc, k, j, loc2));
    __stcs(&bf.rec[2u * idx + 1u], make_uint4((u32)f, (u32)(f >> 32), 0u, 0u));
    const u64 key = NS_STREAM_KEY(k - bf.k_base, f);
    if (bf.key_shift) __stcs((u32 *)bf.rec_key + idx, (u32)(key >> bf.key_shift));
    else __stcs((unsigned long long *)&bf.rec_key[idx], (unsigned long long)key);
}
// the sentinel key of a reserved but unused ring slot: all ones (sorts last, dropped)
__device__ __forceinline__ void store_sentinel(const SimBuffers &bf, u32 idx) {
    if (bf.key_shift) ((u32 *)bf.rec_key)[idx] = ~0u; else bf.rec_key[idx] = ~0ull;
}
__device__ __forceinline__ void record_event(const SimBuffers &bf, u32 loc, u32 k, u32 j, u64 f, u32 loc2) {
    const u32 mask = __activemask();
    const u32 lane = threadIdx.x & 31u;
    const int leader = __ffs(mask) - 1;
    u32 base = 0;
    if ((int)lane == leader) base = atomicAdd(&bf.ctr->n_rec, (u32)__popc(mask));
    base = __shfl_sync(mask, base, leader);
    const u32 idx = base + __popc(mask & lanemask_lt());
    if (idx < bf.rec_cap) store_record(bf, idx, loc, k, j, f, loc2);
}

// ---- approximate event times: the search filter of both simulate kernels (exponential sampler) ----------------------------------------------------
// The decisions of the event-time search ("T >= 2^48" and "T > f_last") are comparisons of partial sums of
// -ln(U_i)/mu. The kernels evaluate them in binary32 from the top 32 bits of each draw: A = (32 - lg2(hi)) * ln2 / mu.
// |A_j - T_j| is bounded ("filter"): a comparison further than the margin from equality has the same outcome as
// the fixed-point comparison of 2.4, anything closer (or a draw with hi < 2^20) is "ambiguous" and the round is redone with
// the exact arithmetic. Exact offsets are needed for records only and are recomputed from the event identity (loc, k, j):
// T(loc, k, j) is a pure function of it (exact_offset).
#define NS_LN2F 0.69314718f
#define NS_MARGIN 6.1035156e-05f                     // 2^-14, times (1 + 1/mu)
// volatile: stays after the table gathers of slot A in issue order (the gathers have the longest latency and go first)
__device__ __forceinline__ float lg2_approx(float x) { float y; asm volatile("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
// 1/mu = Cm * 2^-(24 + sh) as binary32 (T = (E * Cm) >> (32 + sh) with E in Q8.56, T in Q16.48)
__device__ __forceinline__ float rate_to_float(u32 Cm, u32 sh) { return __uint2float_rz(Cm) * __uint_as_float((103u - sh) << 23); }
__device__ __forceinline__ float approx_exp_time(u32 draw_hi, float ln2_over_mu) {
    return (32.0f - lg2_approx(__uint2float_rz(draw_hi))) * ln2_over_mu;
}

// (Cm, sh) of the cell that holds indexed location loc
template <bool PERCELL>
__device__ __forceinline__ uint2 rate_of_loc(const ScenarioDev &sc, u32 loc) {
    if (!PERCELL) return make_uint2(sc.Cm_u, sc.sh_u);
    return __ldg(&sc.scale[cell_of_loc(sc, loc)]);
}
// exact offset T of the event (loc, k, j): the sum of the first j scaled draws of the stream primed on (loc, k)
__device__ __forceinline__ u64 exact_offset(const SeedKey &key, const SmemTables &smt, u32 loc, u32 k, u32 j, u32 Cm, u32 sh) {
    u64 X = prime(key, loc, k), T = 0;
    for (u32 i = 0; i < j; ++i) { X += NS_GAMMA; T += scale_exp(neglog(draw_time(X), smt), Cm, sh); }
    return T;
}
// out-of-line variants for the per-lane kernel, where these rare paths must not cost registers
__device__ __noinline__ u64 exact_offset_nl(SeedKey key, u32 q_addr, u32 a_addr, u32 loc, u32 k, u32 j, u32 Cm, u32 sh) {
    SmemTables smt; smt.q = q_addr; smt.a = a_addr; smt.tg = smt.g2 = smt.pc = smt.pg = 0;
    return exact_offset(key, smt, loc, k, j, Cm, sh);
}
// exact offset of the event (loc, k, j) with the rate of the cell that holds loc (explicit kinds with per-cell turnover)
__device__ __noinline__ u64 exact_offset_of_loc_nl(SeedKey key, u32 q_addr, u32 a_addr, const u32 *prefix, const uint2 *scale, u32 ncells, u32 uniform_deme,
                                                   u32 loc, u32 k, u32 j) {
    u32 c;
    if (uniform_deme) c = loc / uniform_deme;
    else { u32 lo = 0, hi = ncells; while (hi - lo > 1) { u32 mid = lo + ((hi - lo) >> 1); if (prefix[mid] <= loc) lo = mid; else hi = mid; } c = lo; }
    const uint2 cs = __ldg(&scale[c]);
    SmemTables smt; smt.q = q_addr; smt.a = a_addr; smt.tg = smt.g2 = smt.pc = smt.pg = 0;
    return exact_offset(key, smt, loc, k, j, cs.x, cs.y);
}

// phase choice of a pass: SEARCH while n_event * WE <= n_search * WS. Measured on C5 MODE-T: 1:1 (the majority phase) 2.92e10
// events/s, 1:2 (weighted by the cost of a pass: an event pass is about twice a search pass) 2.83e10
#ifndef NS_PHASE_WE
#define NS_PHASE_WE 1u
#define NS_PHASE_WS 1u
#endif
#define NS_COOP_LANES 8u       // cooperative resampling when a warp of an exhausted queue holds at most this many lineages
#define NS_ST_IDLE 0u
#define NS_ST_SEARCH 1u     // needs draws of the event-time search (re-primes first when `need_prime`)
#define NS_ST_EVENT 2u      // event (loc, k, j) found at offset T: `att` dispersal attempts rejected so far

// SAMP: 0 = exponential event-time sampler, 1 = Poisson / order statistics (2.7)
// REC: also append every executed event to the stream ring (NEXT-3)
template <int KIND, bool DEDUP, bool PERCELL, int SAMP, bool REC, bool COMPACT>
__global__ void __launch_bounds__(256, 5) simulate_kernel(const ScenarioDev sc, const SimBuffers bf, const EpochArgs ep) {
    __shared__ unsigned short sQ[SAMP == 0 ? 512 : 256];      // SAMP 1: the Poisson guide
    __shared__ u64 sA[SAMP == 0 ? 512 : 256];                 // SAMP 1: the Poisson cdf thresholds
    __shared__ u32 sG[KIND == 3 ? 1024 : 1];
    __shared__ uint2 sG2[KIND == 3 ? NS_G2_LEN : 1];
    if (SAMP == 0) for (u32 i = threadIdx.x; i < 512; i += blockDim.x) { sQ[i] = NEGLOG_Q_DEV[i]; sA[i] = NEGLOG_A_DEV[i]; }
    else poisson_stage(sc, sA, sQ);
    if (KIND == 3) gauss_stage(sc, sG, sG2);
    __syncthreads();
    GaussLut gl; gl.tg = smem_addr(sG); gl.g2 = smem_addr(sG2); gl.R = sc.R;
    SmemTables smt; smt.q = smem_addr(sQ); smt.a = smem_addr(sA); smt.tg = gl.tg; smt.g2 = gl.g2; smt.pc = smt.a; smt.pg = smt.q;

    const u32 lane = threadIdx.x & 31u;
    const u32 on_mask = ep.lanes_per_warp >= 32u ? 0xFFFFFFFFu : ((1u << ep.lanes_per_warp) - 1u);   // lanes that hold lineages

    // lineage state (registers)
    u32 st = NS_ST_IDLE, att = 0;
    bool need_prime = false, exhausted = false;
    u32 id = 0, loc = 0, cell = 0, k = 0, steps = 0, j = 0, Cm = sc.Cm_u, sh = sc.sh_u;
    i64 f_last = -1;
    u64 X = 0, T = 0;
    // search filter (FILT: exponential sampler without the event stream): the partial sum `a` and the lower bound `fa_last` are
    // binary32 (see approx_exp_time); exact offsets are recomputed from the event identity where a record or an ambiguous comparison
    // needs them. (e_loc, k, e_j) = the last executed event, whose offset is the exact lower bound while fa_last >= 0.
    constexpr bool FILT = (SAMP == 0) && !REC;
    float a = 0.0f, fa_last = -1.0f, lnmu = NS_LN2F * rate_to_float(sc.Cm_u, sc.sh_u);
    u32 e_loc = 0xFFFFFFFFu, e_j = 0;
    const float margin = sc.margin;
    u32 c_events = 0, c_culled = 0, c_resamples = 0;   // per-thread counters, reduced at the end
    u32 rec_next = 0, rec_left = 0;                    // REC: the warp's reserved ring slots (warp-uniform)

    for (;;) {
        // ---- S4: refill idle lanes from the device work queue (one atomic per warp) -----------------
        u32 bs = __ballot_sync(NS_FULL, st == NS_ST_SEARCH);
        const u32 be = __ballot_sync(NS_FULL, st == NS_ST_EVENT);
        const u32 need = on_mask & ~(bs | be);                 // idle lanes that may hold a lineage
        if (need != 0u && !exhausted) {
            u32 cnt = __popc(need), base = 0;
            if (lane == 0) base = atomicAdd(&bf.ctr->q_head, cnt);
            base = __shfl_sync(NS_FULL, base, 0);
            if ((need >> lane) & 1u) {
                u32 idx = base + __popc(need & lanemask_lt());
                if (idx < bf.q_in_count) {
                    uint4 e = bf.q_in[idx];
                    id = e.x; loc = e.y; cell = e.z; steps = e.w;
                    k = ep.k_start; f_last = -1; fa_last = -1.0f; need_prime = true; st = NS_ST_SEARCH;
                }
            }
            exhausted = (base + cnt >= bf.q_in_count);
            bs = __ballot_sync(NS_FULL, st == NS_ST_SEARCH);
        }
        const u32 n_search = __popc(bs), n_event = __popc(be);
        if ((n_search | n_event) == 0u) break;
        bool rec_now = false;          // REC: this lane executed an event in this pass (its k, j, T are unchanged until the next pass)
        u32 r_loc = 0, r_l2 = 0;

        if (n_event * NS_PHASE_WE <= n_search * NS_PHASE_WS) {
            // ======== SEARCH phase ======================================================================
            // S1a: (re-)prime on (loc, k); pause at the epoch horizon
            bool pause = false;
            if (st == NS_ST_SEARCH && need_prime) {
                if (k == ep.k_stop) {
                    pause = true;
                } else {
                    X = prime(ep.key, loc, k);
                    T = 0; a = 0.0f; j = 0; need_prime = false;
                    if (SAMP == 0) {
                        if (PERCELL) {
                            uint2 cs = __ldg(&sc.scale[KIND == 3 ? xy_index(sc, cell) : cell]); Cm = cs.x; sh = cs.y;
                            if (FILT) lnmu = NS_LN2F * rate_to_float(Cm, sh);
                        }
                    } else {   // sh = number of points of this interval, Cm = thinning threshold of the cell, att = best point so far
                        sh = poisson_count(X, smt); att = 0;
                        if (PERCELL) Cm = __ldg(&sc.thin[KIND == 3 ? xy_index(sc, cell) : cell]);
                    }
                }
            }
            {   // survivors of this epoch go to the output queue (warp-aggregated append)
                u32 pm = __ballot_sync(NS_FULL, pause);
                if (pm) {
                    u32 base = 0;
                    if (lane == (u32)(__ffs(pm) - 1)) base = atomicAdd(&bf.ctr->q_out, __popc(pm));
                    base = __shfl_sync(NS_FULL, base, __ffs(pm) - 1);
                    if (pause) {
                        bf.q_out[base + __popc(pm & lanemask_lt())] = make_uint4(id, loc, cell, steps);
                        st = NS_ST_IDLE;
                    }
                }
            }
            if (SAMP == 1 && st == NS_ST_SEARCH) {
                // S1b (Poisson): scan the interval's points; keep the earliest one after f_last (ties: smallest i)
#pragma unroll 1
                for (u32 q = 0; q < 4u && j < sh; ++q) {   // up to four points per pass: amortises the phase scheduling
                    j += 1; X += NS_GAMMA;
                    const u64 f = poisson_offset(X);
                    if ((i64)f > f_last && (att == 0u || f < T)) {         // a better candidate: only now pay for the thinning draw
                        if (!PERCELL || poisson_kept(X, Cm)) { T = f; att = j; }
                    }
                }
                if (j >= sh) {                             // interval scanned
                    if (att) { X -= (u64)(sh - att) * NS_GAMMA; j = att; att = 0; st = NS_ST_EVENT; }
                    else if (k == 0xFFFFFFFFu) { atomicMax(&bf.ctr->error, 3u); st = NS_ST_IDLE; }
                    else { k += 1; f_last = -1; need_prime = true; }
                }
            }
            if (SAMP == 0 && !FILT && st == NS_ST_SEARCH) {
                // S1b: one exponential draw of the event-time search
                j += 1; X += NS_GAMMA;
                T += scale_exp(neglog(draw_time(X), smt), Cm, sh);
                if (T >= NS_TWO48) {                       // interval exhausted: cross and re-prime (L719, L727)
                    if (k == 0xFFFFFFFFu) { atomicMax(&bf.ctr->error, 3u); st = NS_ST_IDLE; }
                    else { k += 1; f_last = -1; need_prime = true; }
                } else if ((i64)T > f_last) {              // strictly later than the last event (L729): the next event
                    st = NS_ST_EVENT; att = 0;
                }
            }
            if (FILT && st == NS_ST_SEARCH) {
                // S1b: one exponential draw of the event-time search, decided in binary32 where the outcome is certain
                j += 1; X += NS_GAMMA;
                const u32 hh = (u32)(draw_time(X) >> 32);
                a += approx_exp_time(hh, lnmu);
                bool outs = a > 1.0f + margin;                                           // T >= 2^48: interval exhausted
                const bool ins = a < 1.0f - margin;
                bool aft = a > fa_last + 2.0f * margin, bef = a < fa_last - 2.0f * margin;   // T > f_last (strictly later, L729)
                if (loc == e_loc && fa_last >= 0.0f) { aft = j > e_j; bef = !aft; }      // same stream as the last event: by ordinal
                // not decided here: coarse logarithm (hi < 2^20), an increment that may round to zero (hi >= 2^32 - 2^8), a partial
                // sum of many terms, a comparison inside the margin
                if ((hh - (1u << 20) >= 0xFFEFFF00u) || j > 32u || !(ins || outs) || (ins && !(aft || bef))) {
                    const u64 Tx = exact_offset_nl(ep.key, smt.q, smt.a, loc, k, j, Cm, sh);
                    i64 fl = -1;
                    if (fa_last >= 0.0f)
                        fl = PERCELL ? (i64)exact_offset_of_loc_nl(ep.key, smt.q, smt.a, sc.prefix, sc.scale, sc.ncells, sc.uniform_deme, e_loc, k, e_j)
                                     : (i64)exact_offset_nl(ep.key, smt.q, smt.a, e_loc, k, e_j, Cm, sh);
                    outs = Tx >= NS_TWO48; aft = (i64)Tx > fl;
                    a = (float)Tx * 0x1p-48f;
                }
                if (outs) {                                // interval exhausted: cross and re-prime (L719, L727)
                    if (k == 0xFFFFFFFFu) { atomicMax(&bf.ctr->error, 3u); st = NS_ST_IDLE; }
                    else { k += 1; fa_last = -1.0f; need_prime = true; }
                } else if (aft) {                          // the next event
                    st = NS_ST_EVENT; att = 0;
                }
            }
        } else if (st == NS_ST_EVENT) {
            // ======== EVENT phase: event (loc, k, j) at offset T ==========================================
            bool culled = false, speciates = false;
            uint4 old = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
            if (att == 0) {
                // S5: duplicate-culling cache keyed on the full event identity; the 128-bit exchange is issued first
                // and consumed after the (side-effect free) speciation and dispersal draws of this pass
                if (DEDUP) {
                    const u32 h = cache_hash(X);
                    if (cache_probes(h, ep.probe_mask)) old = atomic_exch_128(&bf.cache[h & bf.cache_mask], make_uint4(loc, k, j, id));
                }
                // S2: speciation test on the event's SPEC lane (local community of the implicit model: nu = 0, L1830)
                speciates = !(KIND == 1 && cell == 0) && bern(draw_spec(X), ep.thr_nu);
            }
            // S3: one dispersal attempt (KIND 0..2 always accept)
            u32 loc2 = loc, cell2 = cell;
            bool accept = true;
            if (KIND != 3) {
                u32 rs = 0;
                disperse<KIND>(sc, ep.thr_m, X, cell, loc2, cell2, gl, rs);
            } else {
                const u64 x = draw_disp(X, att);
                const u32 xx = wrap_add(cell & 0xFFFFu, gauss_disp(gl, (u32)(x >> 32)), sc.width);
                const u32 yy = wrap_add(cell >> 16, gauss_disp(gl, (u32)x), sc.height);
                u32 d, pfx = 0;
                if (COMPACT) {   // deme and prefix of the target from one 8-byte read of the compact habitat table
                    const uint2 hb = __ldg(&sc.hab64[hab64_index(sc, xx, yy)]);
                    const u32 bit = 1u << (xx & 31u);
                    d = (hb.x & bit) ? sc.compact_deme : 0u;
                    pfx = hb.y + sc.compact_deme * (u32)__popc(hb.x & (bit - 1u));
                } else {
                    d = cell_deme_at(sc, yy * sc.width + xx, k);
                }
                accept = d > 0u;
                if (accept) {
                    cell2 = (yy << 16) | xx;
                    if (!COMPACT) pfx = cell_prefix(sc, yy * sc.width + xx);
                    loc2 = pfx + ((d == 1u) ? 0u : mulhi64_u32(draw_index(X), d));
                }
            }
            if (att == 0) {
                if (DEDUP) culled = old.x == loc && old.y == k && old.z == j && old.w != id;
                if (FILT && (culled || speciates)) T = exact_offset_nl(ep.key, smt.q, smt.a, loc, k, j, Cm, sh);   // the record's exact offset
                if (culled) {
                    // another lineage executed this event: identical future (L687, L697) -> cull, link to it
                    bf.parent[id] = old.w; bf.state[id] = 2;
                    bf.term_loc[id] = loc; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = T; bf.steps[id] = steps;
                    c_culled++; st = NS_ST_IDLE;
                } else {
                    f_last = (i64)T; steps++; c_events++;
                    if (FILT) { fa_last = a; e_loc = loc; e_j = j; }
                    if (speciates) {
                        bf.state[id] = 1;
                        bf.term_loc[id] = loc; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = T; bf.steps[id] = steps;
                        bf.spec_ring[atomicAdd(&bf.ctr->n_spec, 1u)] = id;
                        atomicMax(&bf.ctr->j_max, j);
                        if (REC) { rec_now = true; r_loc = loc; r_l2 = 0xFFFFFFFFu; }
                        st = NS_ST_IDLE;
                    }
                }
            }
            if (st == NS_ST_EVENT) {
                if (accept) {
                    if (REC) { rec_now = true; r_loc = loc; r_l2 = loc2; }
                    loc = loc2; cell = cell2; need_prime = true; st = NS_ST_SEARCH;
                    if (ep.max_steps && steps >= ep.max_steps) {
                        if (FILT) T = exact_offset_nl(ep.key, smt.q, smt.a, e_loc, k, j, Cm, sh);   // (Cm, sh) are still the origin's
                        bf.state[id] = 3;
                        bf.term_loc[id] = loc; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = T; bf.steps[id] = steps;
                        st = NS_ST_IDLE;
                    }
                } else {
                    c_resamples++;
                    if (++att >= NS_MAX_RESAMPLE) { atomicMax(&bf.ctr->error, 3u); st = NS_ST_IDLE; }
                }
            }
        }
        if (KIND == 3 && !REC && exhausted && n_search + n_event <= NS_COOP_LANES) {
            // Cooperative resampling at the ragged end of an epoch: the queue is empty and this warp holds only a few lineages. One that
            // has just had a dispersal attempt rejected (a sparsely inhabited neighbourhood: tens of attempts per event, one pass each)
            // gets its next 32 attempts evaluated by the whole warp. Same draws, same first accepted attempt (R16): identical results.
            u32 em = __ballot_sync(NS_FULL, st == NS_ST_EVENT && att >= 1u);
            while (em) {
                const int L = __ffs(em) - 1;
                em &= em - 1u;
                const u64 bX = __shfl_sync(NS_FULL, X, L);
                const u32 bcell = __shfl_sync(NS_FULL, cell, L), batt = __shfl_sync(NS_FULL, att, L), bk = __shfl_sync(NS_FULL, k, L);
                const u64 x = draw_disp(bX, batt + lane);
                const u32 xx = wrap_add(bcell & 0xFFFFu, gauss_disp(gl, (u32)(x >> 32)), sc.width);
                const u32 yy = wrap_add(bcell >> 16, gauss_disp(gl, (u32)x), sc.height);
                u32 d, pfx;
                if (COMPACT) {
                    const uint2 hb = __ldg(&sc.hab64[hab64_index(sc, xx, yy)]);
                    const u32 bit = 1u << (xx & 31u);
                    d = (hb.x & bit) ? sc.compact_deme : 0u;
                    pfx = hb.y + sc.compact_deme * (u32)__popc(hb.x & (bit - 1u));
                } else {
                    d = cell_deme_at(sc, yy * sc.width + xx, bk);
                    pfx = d ? cell_prefix(sc, yy * sc.width + xx) : 0u;
                }
                const u32 okm = __ballot_sync(NS_FULL, d > 0u);
                const int fa = okm ? __ffs(okm) - 1 : 0;
                const u32 d_f = __shfl_sync(NS_FULL, d, fa), pfx_f = __shfl_sync(NS_FULL, pfx, fa), c2_f = __shfl_sync(NS_FULL, (yy << 16) | xx, fa);
                if ((int)lane == L) {
                    if (okm) {
                        c_resamples += (u32)fa;
                        loc = pfx_f + ((d_f == 1u) ? 0u : mulhi64_u32(draw_index(X), d_f)); cell = c2_f; need_prime = true; st = NS_ST_SEARCH;
                        if (ep.max_steps && steps >= ep.max_steps) {
                            if (FILT) T = exact_offset_nl(ep.key, smt.q, smt.a, e_loc, k, j, Cm, sh);   // (Cm, sh) are still the origin's
                            bf.state[id] = 3;
                            bf.term_loc[id] = loc; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = T; bf.steps[id] = steps;
                            st = NS_ST_IDLE;
                        }
                    } else {
                        c_resamples += 32u; att += 32u;
                        if (att >= NS_MAX_RESAMPLE) { atomicMax(&bf.ctr->error, 3u); st = NS_ST_IDLE; }
                    }
                }
            }
        }
        if (REC) {
            // The pass's events go to the stream ring from a convergent point: ring slots come out of a chunk the WARP reserved
            // (one atomic on the shared counter per chunk, not per pass: with every warp adding to one address for every few
            // events the counter was the bottleneck of the recording run); a chunk's unused end gets sentinel keys.
            const u32 rm = __ballot_sync(NS_FULL, rec_now);
            if (rm) {
                const u32 cnt = __popc(rm);
                if (rec_left < cnt) {
                    if (lane < rec_left) store_sentinel(bf, rec_next + lane);      // rec_left < cnt <= 32
                    const u32 take = ep.rec_chunk >= 64u ? ep.rec_chunk : cnt;     // small rings: exact reservations
                    u32 base = 0;
                    if (lane == 0) base = atomicAdd(&bf.ctr->n_rec, take);
                    rec_next = __shfl_sync(NS_FULL, base, 0); rec_left = take;
                }
                const u32 idx = rec_next + __popc(rm & lanemask_lt());
                if (rec_now && idx < bf.rec_cap) store_record(bf, idx, r_loc, k, j, T, r_l2);
                rec_next += cnt; rec_left -= cnt;
            }
        }
    }
    if (REC) for (u32 q = lane; q < rec_left; q += 32u) if (rec_next + q < bf.rec_cap) store_sentinel(bf, rec_next + q);   // the last chunk's unused end
    // reduce the per-thread counters: warp shuffle, then one atomic per warp
    unsigned long long r_events = c_events, r_culled = c_culled, r_resamples = c_resamples;
    for (int o = 16; o; o >>= 1) {
        r_events += __shfl_down_sync(NS_FULL, r_events, o);
        r_culled += __shfl_down_sync(NS_FULL, r_culled, o);
        r_resamples += __shfl_down_sync(NS_FULL, r_resamples, o);
    }
    if (lane == 0) {
        if (r_events) atomicAdd((unsigned long long *)&bf.ctr->n_events, r_events);
        if (r_culled) atomicAdd((unsigned long long *)&bf.ctr->n_culled, r_culled);
        if (r_resamples) atomicAdd((unsigned long long *)&bf.ctr->resamples, r_resamples);
    }
}

}  // namespace necsim
