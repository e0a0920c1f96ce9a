// tail_kernel.cuh -- low-latency simulate kernel for the sequential tail: ONE lineage per warp.
//
// At low nu the last lineages are serial chains of ~1/nu events each ("its curve
// never flattens"); with a few thousand lineages left the machine is bound by the latency of one event, not by
// throughput. Every draw is a pure function of its key (seed, loc, k, j, lane) -- PAPER.md 5.2.1, L693-707 --
// so the 32 lanes of a warp may evaluate candidate draws of ONE lineage speculatively and in parallel; the
// result is identical by construction (tests/test_gpu_invariance.py runs both kernels on the same inputs):
//   - candidates: lanes 0..15 hold the points j = 1..16 of interval k (a segmented prefix sum gives the partial
//     sums T_j), lanes 16..31 the FIRST point of intervals k+1..k+16 (the event if interval k is exhausted: a
//     fresh interval's first point is its next event, L719-729);
//   - once the winning candidate is known, ONE hash evaluation across the lanes yields all the event's draws: lane 0
//     the speciation draw, lane 1 the index draw, lane 2 the migration draw, lanes 3..31 the dispersal attempts
//     r = 0..28 (R16), each with its habitat / prefix / turnover-scale gathers; a ballot picks the first accepted;
//   - the duplicate-culling exchange of an event is issued when the event is selected and consumed one event
//     later (never after another cache insertion: an unconfirmed lineage must not publish entries).
#pragma once
#include "sim_kernel.cuh"

namespace necsim {

#define NS_REC_CHUNK 64u           // event-stream ring slots a warp reserves at a time
#define NS_TAIL_ATTEMPTS 29u      // dispersal attempts evaluated per pass (lanes 3..31)


// one level of the inclusive prefix sum over 16-lane segments: T += T of the lane `o` below, where that lane is in the
// same segment (the shuffle's own predicate says so): 2 SHFL + 2 predicated adds
__device__ __forceinline__ void seg16_scan_step(u32 &lo, u32 &hi, u32 o) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        ".reg .b32 tl, th;\n\t"
        "shfl.sync.up.b32 tl|p, %0, %2, 0x1000, 0xffffffff;\n\t"
        "shfl.sync.up.b32 th, %1, %2, 0x1000, 0xffffffff;\n\t"
        "@p add.cc.u32 %0, %0, tl;\n\t"
        "@p addc.u32 %1, %1, th;\n\t"
        "}"
        : "+r"(lo), "+r"(hi)
        : "r"(o));
}

// per-cell rate data: exponential sampler -> (Cm, sh) of 1/(lambda dt); Poisson sampler -> (thinning threshold, unused)
template <int SAMP>
__device__ __forceinline__ uint2 load_rate(const ScenarioDev &sc, u32 idx) {
    if (SAMP == 0) return __ldg(&sc.scale[idx]);
    return make_uint2(__ldg(&sc.thin[idx]), 0u);
}

// Gathers of one dispersal target, issued back to back (volatile: kept in this order): prefix and rate first, the habitat
// byte last, so that the first instruction that needs the habitat byte waits for all three round trips at once.
__device__ __forceinline__ u32 ldg_u32_ordered(const u32 *p) { u32 v; asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(p)); return v; }
__device__ __forceinline__ u32 ldg_u8_ordered(const uint8_t *p) { u32 v; asm volatile("ld.global.nc.u8 %0, [%1];" : "=r"(v) : "l"(p)); return v; }
__device__ __forceinline__ uint2 ldg_v2_ordered(const uint2 *p) {
    uint2 v; asm volatile("ld.global.nc.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p)); return v;
}

// index of the lowest set bit of m != 0: isolate it and take its position (one FLO; __ffs costs BREV + FLO, two trips
// through the quarter-rate unit on a chain where every cycle counts)
__device__ __forceinline__ int first_bit(u32 m) {
    u32 r;
    asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(m & (0u - m)));
    return (int)r;
}

__device__ __forceinline__ u64 shfl_xor_u64(u64 v, int m) { return __shfl_xor_sync(NS_FULL, v, m); }

// Poisson sampler, one search round of one lineage across the warp: lanes 0..15 the points 1..16 of
// interval k, lanes 16..23 / 24..31 the points 1..8 of intervals k+1 / k+2. A butterfly min over (offset, ordinal) keys
// finds the earliest existing point after f_last in the first non-empty interval. Returns true with (k, j, Te, Xe) set;
// false after advancing k past intervals without a next event (the caller loops).
template <bool PERCELL>
__device__ __forceinline__ bool tail_search_poisson(const SeedKey &key, const SmemTables &smt, u32 lane, u32 loc, u32 &k, i64 &f_last,
                                                    u32 k_stop, u32 thin, u32 &j, u64 &Te, u64 &Xe) {
    const u32 seg = lane < 16u ? 0u : (lane < 24u ? 1u : 2u);
    const u32 i = (lane < 16u ? lane : (lane & 7u)) + 1u;
    const u64 kk64 = (u64)k + seg;
    const bool kvalid = kk64 < (u64)k_stop;
    const u64 s = prime(key, loc, (u32)kk64);
    const u64 X = s + (u64)i * NS_GAMMA;
    // the count, offset and thinning draws of this lane's point are independent: evaluated side by side
    u64 hc, hf, ht = 0;
    if (PERCELL) hashF3(s ^ NS_L_COUNT, X, X ^ NS_L_THIN, hc, hf, ht);
    else hashF2(s ^ NS_L_COUNT, X, hc, hf);
    const u32 N = poisson_count_of(hc, smt);
    const u64 f = hf >> 16;
    if (__ballot_sync(NS_FULL, kvalid && N > (seg ? 8u : 16u))) {
        // more points than lanes somewhere (large mu): scan interval k one point at a time (every lane the same)
        const u64 s0 = __shfl_sync(NS_FULL, s, 0);
        const u32 N0 = __shfl_sync(NS_FULL, N, 0);
        u32 bi = 0; u64 bf = 0, Xi = s0;
        for (u32 q = 1; q <= N0; ++q) {
            Xi += NS_GAMMA;
            const u64 fq = poisson_offset(Xi);
            if (PERCELL && !poisson_kept(Xi, thin)) continue;
            if ((i64)fq > f_last && (bi == 0u || fq < bf)) { bi = q; bf = fq; }
        }
        if (!bi) { k += 1u; f_last = -1; return false; }
        j = bi; Te = bf; Xe = s0 + (u64)bi * NS_GAMMA;
        return true;
    }
    bool ok = kvalid && i <= N && (seg != 0u || (i64)f > f_last);
    if (PERCELL) ok = ok && (thin == 0xFFFFFFFFu || (u32)ht < thin);
    u64 m = ok ? ((f << 8) | (u64)i) : ~0ull;
    m = min(m, shfl_xor_u64(m, 1)); m = min(m, shfl_xor_u64(m, 2)); m = min(m, shfl_xor_u64(m, 4));
    const u64 m16 = min(m, shfl_xor_u64(m, 8));
    const u64 m0 = __shfl_sync(NS_FULL, m16, 0), m1 = __shfl_sync(NS_FULL, m, 16), m2 = __shfl_sync(NS_FULL, m, 24);
    u64 best; u32 dk, base;
    if (m0 != ~0ull) { best = m0; dk = 0u; base = 0u; }
    else if (m1 != ~0ull) { best = m1; dk = 1u; base = 16u; }
    else if (m2 != ~0ull) { best = m2; dk = 2u; base = 24u; }
    else {   // no next event in the (up to three) intervals before the horizon
        const u32 gap = k_stop - k;
        k += gap < 3u ? gap : 3u; f_last = -1;
        return false;
    }
    j = (u32)best & 255u; Te = best >> 8; k += dk;
    Xe = __shfl_sync(NS_FULL, X, (int)(base + j - 1u));
    return true;
}

template <int KIND, bool DEDUP, bool PERCELL, int SAMP, bool REC>
__global__ void __launch_bounds__(256) tail_kernel(const ScenarioDev sc, const SimBuffers bf, const EpochArgs ep) {
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

    u32 lane;
    asm volatile("mov.u32 %0, %%laneid;" : "=r"(lane));                // opaque: kept in a register, not re-read per use
    const u32 half = lane >> 4, sub = lane & 15u;
    const u32 jj = half ? 1u : sub + 1u;                               // ordinal of this lane's candidate point
    const u64 cand_add = (u64)jj * NS_GAMMA;                           // stream position of the candidate: s + jj * GAMMA
    // event draws, one per lane: draw = F((X ^ lane_xor) + lane_add)
    const u64 lane_xor = lane == 0 ? NS_L_SPEC : lane == 1 ? NS_L_INDEX : lane == 2 ? NS_L_MIGR : NS_L_DISP;
    const u32 att_lane = lane >= 3u ? lane - 3u : 0u;                  // dispersal attempt of this lane within a pass
    const u64 att_add = (u64)att_lane * NS_GAMMA;
    unsigned long long c_events = 0, c_culled = 0, c_resamples = 0;   // warp-uniform
    // event-stream ring (REC): the warp reserves ep.rec_chunk (<= NS_REC_CHUNK) slots at a time, so that it waits for an atomic's return once per
    // chunk and not once per event; slots left over at the end are filled with sentinels (k = k_stop, which no event of the epoch has) the host-side pass drops
    u32 rec_next = 0, rec_left = 0;
    auto record = [&](u32 r_loc, u32 r_k, u32 r_j, u64 r_f, u32 r_l2) {   // lane 0 only
        if (rec_left == 0u) { rec_next = atomicAdd(&bf.ctr->n_rec, ep.rec_chunk); rec_left = ep.rec_chunk; }
        const u32 ri = rec_next++; --rec_left;
        if (ri < bf.rec_cap) { bf.rec_loc[ri] = r_loc; bf.rec_k[ri] = r_k; bf.rec_j[ri] = r_j; bf.rec_f[ri] = r_f; bf.rec_loc2[ri] = r_l2; }
    };

    for (;;) {
        // ---- S4: one queue entry per warp --------------------------------------------------------------
        u32 qi = 0;
        if (lane == 0) qi = atomicAdd(&bf.ctr->q_head, 1u);
        qi = __shfl_sync(NS_FULL, qi, 0);
        if (qi >= bf.q_in_count) break;
        const uint4 qe = bf.q_in[qi];
        const u32 id = qe.x;
        u32 loc = qe.y, cell = qe.z, steps = qe.w, k = ep.k_start, Cm = sc.Cm_u, sh = sc.sh_u;
        i64 f_last = -1;
        if (PERCELL) { uint2 cs = load_rate<SAMP>(sc, KIND == 3 ? xy_index(sc, cell) : cell); Cm = cs.x; sh = cs.y; }
        // pending duplicate check: the exchange of the last probing event (lane 0 holds its result)
        bool pend = false;
        u64 pold_lo = ~0ull, pold_hi = ~0ull;
        u32 p_loc = 0, p_k = 0, p_j = 0, p_l2 = 0;
        u64 p_T = 0;
        // consumes the pending exchange: true = this lineage is a duplicate at the pending event (culled, recorded)
        auto resolve_pending = [&]() -> bool {
            if (!DEDUP || !pend) return false;
            pend = false;
            const u32 ox = __shfl_sync(NS_FULL, (u32)pold_lo, 0), oy = __shfl_sync(NS_FULL, (u32)(pold_lo >> 32), 0);
            const u32 oz = __shfl_sync(NS_FULL, (u32)pold_hi, 0), ow = __shfl_sync(NS_FULL, (u32)(pold_hi >> 32), 0);
            if (ox == p_loc && oy == p_k && oz == p_j && ow != id) {   // another lineage executed it first (L687, L697)
                if (lane == 0) {
                    bf.parent[id] = ow; bf.state[id] = 2;
                    bf.term_loc[id] = p_loc; bf.term_k[id] = p_k; bf.term_j[id] = p_j; bf.term_f[id] = p_T; bf.steps[id] = steps;
                }
                c_culled++;
                return true;
            }
            steps++; c_events++;                                       // the pending event was really executed
            if (REC && lane == 0) record(p_loc, p_k, p_j, p_T, p_l2);
            return false;
        };

        for (;;) {   // one iteration = one search round (+ the event it finds)
            if (k == ep.k_stop) {   // epoch horizon: survivor (unless its last event turns out to be a duplicate)
                if (resolve_pending()) break;
                if (lane == 0) bf.q_out[atomicAdd(&bf.ctr->q_out, 1u)] = make_uint4(id, loc, cell, steps);
                break;
            }
            u32 j;
            u64 Te, Xe;
            if (SAMP == 1) {
                // S1 (Poisson sampler, Cm = thinning threshold of the cell)
                if (!tail_search_poisson<PERCELL>(ep.key, smt, lane, loc, k, f_last, ep.k_stop, Cm, j, Te, Xe)) continue;
            } else {
                // ---- S1: candidate points of the event-time search ---------------------------------------------------
                const u64 kk64 = (u64)k + (half ? (u64)(1u + sub) : 0ull);
                const bool kvalid = kk64 < (u64)ep.k_stop;                // never look at or past the horizon
                u64 X = prime(ep.key, loc, (u32)kk64) + cand_add;
                const u64 T1 = scale_exp(neglog(draw_time(X), smt), Cm, sh);
                // partial sums over each 16-lane half (half 1 keeps its single draws: first points of fresh intervals)
                u32 t_lo = (u32)T1, t_hi = (u32)(T1 >> 32);
                seg16_scan_step(t_lo, t_hi, 1); seg16_scan_step(t_lo, t_hi, 2);
                seg16_scan_step(t_lo, t_hi, 4); seg16_scan_step(t_lo, t_hi, 8);
                const u64 T = half ? T1 : (((u64)t_hi << 32) | t_lo);
                const bool inside = T < NS_TWO48;
                const u32 evm = __ballot_sync(NS_FULL, inside && (half ? kvalid : ((i64)T > f_last)));
                const u32 crm = __ballot_sync(NS_FULL, !inside);
                if (evm & 0xFFFFu) {                       // next event is in interval k
                    const int src = first_bit(evm & 0xFFFFu);
                    j = (u32)src + 1u;
                    Te = __shfl_sync(NS_FULL, T, src); Xe = __shfl_sync(NS_FULL, X, src);
                } else if (crm & 0xFFFFu) {                // interval k exhausted (L719, L727): first non-empty interval after it
                    const u32 gap = ep.k_stop - 1u - k;    // k < k_stop here
                    const u32 nvalid = gap < 16u ? gap : 16u;
                    const u32 hm = evm >> 16;
                    if (!hm) { k = k + 1u + nvalid; f_last = -1; continue; }   // all speculated intervals empty / beyond the horizon
                    const int src = 16 + first_bit(hm);
                    k = k + 1u + (u32)(src - 16); j = 1u;
                    Te = __shfl_sync(NS_FULL, T, src); Xe = __shfl_sync(NS_FULL, X, src);
                } else {
                    // more than 16 points of interval k at or before f_last (large mu): continue the scan one draw at a time
                    u64 Tc = __shfl_sync(NS_FULL, T, 15), Xc = __shfl_sync(NS_FULL, X, 15);
                    u32 jc = 16u;
                    bool found = false;
                    for (;;) {
                        jc += 1u; Xc += NS_GAMMA;
                        Tc += scale_exp(neglog(draw_time(Xc), smt), Cm, sh);
                        if (Tc >= NS_TWO48) break;
                        if ((i64)Tc > f_last) { found = true; break; }
                    }
                    if (!found) { k += 1u; f_last = -1; continue; }
                    j = jc; Te = Tc; Xe = Xc;
                }
            }

            // ---- event (loc, k, j) at offset Te --------------------------------------------------------------
            // S5: the previous probing event's exchange is consumed before this event may publish a cache entry
            if (resolve_pending()) break;
            bool probes = false;
            if (DEDUP) {
                const u32 h = cache_hash(loc, k, j);
                probes = cache_probes(h, ep.probe_mask);
                atomic_exch_128_if(probes && lane == 0, &bf.cache[h & bf.cache_mask], make_uint4(loc, k, j, id), pold_lo, pold_hi);
                if (probes) { p_loc = loc; p_k = k; p_j = j; p_T = Te; pend = true; }
            }
            if (!probes) { steps++; c_events++; }
            // S2 + S3: all draws of the event in one hash evaluation across the lanes
            const u64 xb = Xe ^ lane_xor;
            u64 u = hashF(xb + att_add);
            const bool can_speciate = !(KIND == 1 && cell == 0);      // local community of the implicit model: nu = 0 (L1830)
            const u32 bm = __ballot_sync(NS_FULL, bern(u, lane == 2 ? ep.thr_m : ep.thr_nu));
            const bool speciates = can_speciate && (bm & 1u);
            u32 loc2 = loc, cell2 = cell, Cm2 = Cm, sh2 = sh;
            bool ok = true;
            if (!speciates) {
                if (KIND == 0) {
                    loc2 = mulhi64_u32(__shfl_sync(NS_FULL, u, 3), (u32)sc.n_locations); cell2 = 0;
                } else if (KIND == 1) {
                    const u64 x = __shfl_sync(NS_FULL, u, 3);
                    const bool to_meta = (cell != 0) || (bm & 4u);
                    if (to_meta) { loc2 = sc.J_local + mulhi64_u32(x, sc.J_meta); cell2 = 1; }
                    else { loc2 = mulhi64_u32(x, sc.J_local); cell2 = 0; }
                } else if (KIND == 2) {
                    const u64 x = __shfl_sync(NS_FULL, u, 3), xi = __shfl_sync(NS_FULL, u, 1);
                    const u32 n = sc.ncells, col = __umulhi((u32)(x >> 32), n);
                    const uint2 e = __ldg(&sc.alias[(size_t)cell * n + col]);
                    cell2 = ((u32)x < e.x) ? col : e.y;
                    const u32 d = cell_deme(sc, cell2);
                    loc2 = cell_prefix(sc, cell2) + ((d == 1u) ? 0u : mulhi64_u32(xi, d));
                    if (PERCELL) { const uint2 cs = load_rate<SAMP>(sc, cell2); Cm2 = cs.x; sh2 = cs.y; }
                } else {
                    const u64 xi = __shfl_sync(NS_FULL, u, 1);
                    const u32 x0 = cell & 0xFFFFu, y0 = cell >> 16;
                    ok = false;
                    for (u32 r0 = 0; r0 < NS_MAX_RESAMPLE; r0 += NS_TAIL_ATTEMPTS) {
                        u32 c2 = 0, d = 0, pf = 0;
                        uint2 cs = make_uint2(Cm, sh);
                        if (lane >= 3u) {   // attempt r0 + lane - 3 (R16: redraw the whole (dx, dy) pair)
                            bool e1, e2;
                            int dx = gauss_disp_fast(gl, (u32)(u >> 32), e1), dy = gauss_disp_fast(gl, (u32)u, e2);
                            if (!(e1 && e2)) { dx = gauss_disp(gl, (u32)(u >> 32)); dy = gauss_disp(gl, (u32)u); }   // rare: crowded tail buckets
                            const u32 xx = wrap_add(x0, dx, sc.width);
                            const u32 yy = wrap_add(y0, dy, sc.height);
                            const u32 ci = yy * sc.width + xx;
                            c2 = (yy << 16) | xx;
                            pf = ldg_u32_ordered(&sc.prefix[ci]);           // speculative: same round trip as the habitat test
                            if (PERCELL) {
                                if (SAMP == 0) cs = ldg_v2_ordered(&sc.scale[ci]);
                                else cs.x = ldg_u32_ordered(&sc.thin[ci]), cs.y = 0u;
                            }
                            d = ldg_u8_ordered(&sc.hab8[ci]);
                            if (d == 255u) d = __ldg(&sc.deme32[ci]);
                        }
                        const u32 okm = __ballot_sync(NS_FULL, lane >= 3u && d > 0u);
                        if (okm) {
                            const int w = first_bit(okm);    // first accepted attempt = the sequential algorithm's choice
                            c2 = __shfl_sync(NS_FULL, c2, w); d = __shfl_sync(NS_FULL, d, w); pf = __shfl_sync(NS_FULL, pf, w);
                            if (PERCELL) { Cm2 = __shfl_sync(NS_FULL, cs.x, w); sh2 = __shfl_sync(NS_FULL, cs.y, w); }
                            cell2 = c2;
                            loc2 = pf + ((d == 1u) ? 0u : mulhi64_u32(xi, d));
                            c_resamples += r0 + (u32)w - 3u;
                            ok = true;
                            break;
                        }
                        u = hashF(xb + att_add + (u64)(r0 + NS_TAIL_ATTEMPTS) * NS_GAMMA);   // next 29 attempts
                    }
                }
            }
            if (REC) {   // the event's record: now if it did not probe, else when its exchange is consumed
                const u32 l2 = speciates ? 0xFFFFFFFFu : loc2;
                if (pend) p_l2 = l2;
                else if (lane == 0) record(loc, k, j, Te, l2);
            }
            const u32 steps_e = steps + (pend ? 1u : 0u);              // step count if this event is confirmed
            const bool capped = ep.max_steps && steps_e >= ep.max_steps;
            if (speciates || !ok || capped) {   // terminal: the event's own duplicate check must be known first
                if (resolve_pending()) break;
                if (lane == 0) {
                    if (speciates) {
                        bf.state[id] = 1;
                        bf.term_loc[id] = loc; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = Te; bf.steps[id] = steps;
                        bf.spec_ring[atomicAdd(&bf.ctr->n_spec, 1u)] = id;
                        atomicMax(&bf.ctr->j_max, j);
                    } else if (!ok) {
                        atomicMax(&bf.ctr->error, 3u);
                    } else {
                        bf.state[id] = 3;
                        bf.term_loc[id] = loc2; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = Te; bf.steps[id] = steps;
                    }
                }
                break;
            }
            f_last = (i64)Te; loc = loc2; cell = cell2; Cm = Cm2; sh = sh2;
        }
    }
    if (REC) {   // sentinels into the reserved slots that stayed empty
        const u32 nx = __shfl_sync(NS_FULL, rec_next, 0), lf = __shfl_sync(NS_FULL, rec_left, 0);
        for (u32 q = lane; q < lf; q += 32u) {
            const u32 ri = nx + q;
            if (ri < bf.rec_cap) { bf.rec_loc[ri] = 0xFFFFFFFFu; bf.rec_k[ri] = ep.k_stop; bf.rec_j[ri] = 0xFFFFFFFFu; bf.rec_f[ri] = ~0ull; bf.rec_loc2[ri] = 0xFFFFFFFFu; }
        }
    }
    if (lane == 0) {
        if (c_events) atomicAdd((unsigned long long *)&bf.ctr->n_events, c_events);
        if (c_culled) atomicAdd((unsigned long long *)&bf.ctr->n_culled, c_culled);
        if (c_resamples) atomicAdd((unsigned long long *)&bf.ctr->resamples, c_resamples);
    }
}

}  // namespace necsim
