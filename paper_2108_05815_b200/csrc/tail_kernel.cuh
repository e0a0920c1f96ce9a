// tail_kernel.cuh -- low-latency simulate kernel for the sequential tail: ONE lineage per warp.
//
// At low nu the last lineages are serial chains of ~1/nu events each ("its curve
// never flattens"); with a few thousand lineages left the machine is bound by the latency of one event, not by
// throughput. Every draw is a pure function of its key (seed, loc, k, j, lane) -- PAPER.md 5.2.1, L693-707 --
// so the 32 lanes of a warp may evaluate candidate draws of ONE lineage speculatively and in parallel; the
// result is identical by construction (tests/test_gpu_invariance.py runs both kernels on the same inputs):
//   - candidates: the points j = 1.. of interval k (a prefix sum over the lanes gives the partial sums T_j) and the FIRST
//     point of the following intervals (the event if interval k is exhausted: a fresh interval's first point is its next
//     event, L719-729);
//   - general path, once the winning candidate is known: ONE hash evaluation across the lanes yields all the event's draws: lane 0
//     the speciation draw, lane 1 the index draw, lane 2 the migration draw, lanes 3..31 the dispersal attempts
//     r = 0..28 (R16), each with its habitat / prefix / turnover-scale gathers; a ballot picks the first accepted;
//   - the duplicate-culling exchange of an event is issued when the event is selected and consumed one event
//     later (never after another cache insertion: an unconfirmed lineage must not publish entries).
//
// Exponential sampler, fast path ("speculative round"): the search for the next event and the evaluation of the events it
// may find run SIDE BY SIDE, not one after the other. The draws of a candidate event are a pure function of (seed, loc, k, j)
// and do not depend on its time, so each round the warp evaluates, with two interleaved hash evaluations per lane,
//   8 candidates (lane >> 2): the points j = 1..5 of interval k and the first point of the intervals k+1, k+2, k+3
//                             (99.6 % of the events at mu = 2, measured by simulation; the rest takes the general path)
//   x 4 lanes (lane & 3):     slot A = dispersal attempt r = lane & 3 with its rounded-normal lookups and table gathers,
//                             slot B = the time draw / speciation draw / index draw / migration draw of the candidate.
// While the gathers are in flight the warp computes the logarithms and the partial sums; two ballots pick the event, a third
// the first accepted attempt among the winner's four lanes. The critical path of an event is prime -> hash -> max(gather,
// logarithm + scan) -> select instead of prime -> hash -> logarithm -> scan -> select -> hash -> gather -> select.
// While the ballots pick the winner, every candidate's lanes already prime the stream states of the NEXT round from the candidate's own
// outcome; after the commit they come from the winner's lanes by shuffle. Rounds that are not clean but common are handled without the
// exact path: the first five points all before the bound -> a continuation round over the next five (partial sum carried over); the
// winner's dispersal unsettled (four attempts rejected, or an undetermined target at or before the first accepted one) -> an attempt
// round after the loop that puts 32 attempts of the known event on the lanes. Everything else (ambiguous comparisons, a duplicate, a
// speciation, the step cap, three empty intervals in a row: 0.6 % of the events of C5's tail) falls back to the general code below,
// which recomputes the exact lower bound from the last event's identity (identical results).
#pragma once
#include "sim_kernel.cuh"

namespace necsim {

#define NS_SPEC_NJ 5u              // speculative round: candidates 0..4 = points 1..5 of interval k
#define NS_SPEC_ND 3u              //                    candidates 5..7 = first point of intervals k+1..k+3

#define NS_REC_CHUNK 64u           // event-stream ring slots a warp reserves at a time
#define NS_TAIL_ATTEMPTS 29u      // dispersal attempts evaluated per pass (lanes 3..31)


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

// dispersal target of one attempt of EXPLICIT_GAUSSIAN from (x0, y0) with the draw u: packed cell, deme (0 = not habitat: rejected),
// prefix of the cell, rate data of the cell. The gathers are issued back to back before anything consumes them.
// FAST: no exact rescan of crowded guide buckets (far tails, probability ~ 2^-10): `bad` says that the target is unknown.
template <bool PERCELL, int SAMP, bool COMPACT, bool FAST>
__device__ __forceinline__ void gauss_target(const ScenarioDev &sc, const GaussLut &gl, u32 x0, u32 y0, u64 u, u32 k, u32 &c2, u32 &d, u32 &pf, uint2 &cs, bool &bad) {
    bool e1, e2;
    int dx = gauss_disp_fast(gl, (u32)(u >> 32), e1), dy = gauss_disp_fast(gl, (u32)u, e2);
    bad = !(e1 && e2);
    if (!FAST && bad) { dx = gauss_disp(gl, (u32)(u >> 32)); dy = gauss_disp(gl, (u32)u); }   // rare: crowded tail buckets
    const u32 xx = wrap_add(x0, dx, sc.width);
    const u32 yy = wrap_add(y0, dy, sc.height);
    c2 = (yy << 16) | xx;
    if (COMPACT) {
        const uint2 hb = ldg_v2_ordered(&sc.hab64[hab64_index(sc, xx, yy)]);
        if (PERCELL) {
            const u32 ci = yy * sc.width + xx;
            if (SAMP == 0) cs = ldg_v2_ordered(&sc.scale[ci]);
            else cs.x = ldg_u32_ordered(&sc.thin[ci]), cs.y = 0u;
        }
        const u32 bit = 1u << (xx & 31u);
        d = (hb.x & bit) ? sc.compact_deme : 0u;
        pf = hb.y + sc.compact_deme * (u32)__popc(hb.x & (bit - 1u));
    } else {
        const u32 ci = yy * sc.width + xx;
        pf = ldg_u32_ordered(&sc.prefix[ci]);           // speculative: same round trip as the habitat test
        if (PERCELL) {
            if (SAMP == 0) cs = ldg_v2_ordered(&sc.scale[ci]);
            else cs.x = ldg_u32_ordered(&sc.thin[ci]), cs.y = 0u;
        }
        if (sc.n_eras) d = cell_deme_at(sc, ci, k);         // temporally varying habitat: the map of the event's interval
        else { d = ldg_u8_ordered(&sc.hab8[ci]); if (d == 255u) d = __ldg(&sc.deme32[ci]); }
    }
}

__device__ __forceinline__ uint2 lds_v2_ordered(u32 addr) { uint2 v; asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr)); return v; }
// (x * d) >> 64 for a 32-bit d (see mulhi64_u32), with the two halves of x given
__device__ __forceinline__ u32 mulhi64_u32_parts(u32 xlo, u32 xhi, u32 d) {
    const u64 hi = (u64)xhi * (u64)d + (u64)__umulhi(xlo, d);
    return (u32)(hi >> 32);
}

// Fast round, slot A of one lane (DESIGN.md 2.5 step 2): the dispersal target this lane's draw `ua` leads to, as the complete new
// location: loc2 = prefix[cell'] + index, cell' (packed for EXPLICIT_GAUSSIAN), rate of cell'. acc = the target is habitat (this
// attempt is accepted); bad = the target could not be determined here (crowded guide bucket): the round falls back.
// xi = the index draw of the lane's candidate. Loads are issued before anything consumes them.
template <int KIND, bool PERCELL, bool COMPACT>
__device__ __forceinline__ void fast_slot_a(const ScenarioDev &sc, const GaussLut &gl, u32 sp_q, u32 lane, u32 bm, u32 cell, u32 kc, u64 ua, u32 xi_lo, u32 xi_hi,
                                            u32 &loc2, u32 &c2, uint2 &cs, bool &acc, bool &bad, u32 &tie) {
    bad = false; tie = 0u;
    if (KIND == 0) {
        loc2 = mulhi64_u32(ua, (u32)sc.n_locations); c2 = 0u; acc = sp_q == 0u;
    } else if (KIND == 1) {
        const bool to_meta = (cell != 0) || ((bm >> ((lane & 28u) + 3u)) & 1u);
        loc2 = to_meta ? sc.J_local + mulhi64_u32(ua, sc.J_meta) : mulhi64_u32(ua, sc.J_local);
        c2 = to_meta ? 1u : 0u; acc = sp_q == 0u;
    } else if (KIND == 2) {
        u32 d = 0, pf = 0;
        c2 = 0;
        if (sp_q == 0u) {
            const u32 n = sc.ncells, col = __umulhi((u32)(ua >> 32), n);
            const uint2 e = __ldg(&sc.alias[(size_t)cell * n + col]);
            c2 = ((u32)ua < e.x) ? col : e.y;
            pf = ldg_u32_ordered(&sc.prefix[c2]);
            if (PERCELL) cs = ldg_v2_ordered(&sc.scale[c2]);
            d = ldg_u8_ordered(&sc.hab8[c2]);
            if (d == 255u) d = __ldg(&sc.deme32[c2]);
        }
        acc = d > 0u;
        loc2 = pf + ((d == 1u) ? 0u : mulhi64_u32_parts(xi_lo, xi_hi, d));
    } else {
        // rounded-normal displacement of both axes: the two guide reads back to back, then pos = pos0 + (u >= threshold)
        const u32 ux = (u32)(ua >> 32), uy = (u32)ua;
        const uint2 ex = lds_v2_ordered(gl.g2 + 8u * (ux >> (32 - NS_G2_BITS)));
        const uint2 ey = lds_v2_ordered(gl.g2 + 8u * (uy >> (32 - NS_G2_BITS)));
        bad = ((ex.x | ey.x) >> 16) != 0u;
        // torus (R17): t = coordinate + displacement + size lies in (0, 3 * size); two unsigned minima with t - size bring it into [0, size)
        u32 xx = (ex.x & 0xFFFFu) + ((ex.y <= ux) ? 1u : 0u) + ((cell & 0xFFFFu) + sc.width - (u32)gl.R);
        u32 yy = (ey.x & 0xFFFFu) + ((ey.y <= uy) ? 1u : 0u) + ((cell >> 16) + sc.height - (u32)gl.R);
        xx = min(xx, xx - sc.width); xx = min(xx, xx - sc.width);
        yy = min(yy, yy - sc.height); yy = min(yy, yy - sc.height);
        c2 = (yy << 16) | xx;
        if (COMPACT) {
            const uint2 hb = __ldg(&sc.hab64[hab64_index(sc, xx, yy)]);
            if (PERCELL) cs = __ldg(&sc.scale[yy * sc.width + xx]);
            const u32 D = sc.compact_deme;
            const u32 idx = (D == 1u) ? 0u : mulhi64_u32_parts(xi_lo, xi_hi, D);     // in flight with the gather
            const u32 bit = 1u << (xx & 31u);
            acc = (hb.x & bit) != 0u;
            loc2 = hb.y + D * (u32)__popc(hb.x & (bit - 1u)) + idx;
            tie = hb.x;
        } else {
            const u32 ci = yy * sc.width + xx;
            const u32 pf = ldg_u32_ordered(&sc.prefix[ci]);
            if (PERCELL) cs = ldg_v2_ordered(&sc.scale[ci]);
            u32 d;
            if (sc.n_eras) d = cell_deme_at(sc, ci, kc);    // temporally varying habitat: the map of the candidate's interval
            else { d = ldg_u8_ordered(&sc.hab8[ci]); if (d == 255u) d = __ldg(&sc.deme32[ci]); }
            acc = d > 0u;
            loc2 = pf + ((d == 1u) ? 0u : mulhi64_u32_parts(xi_lo, xi_hi, d));
        }
    }
}

template <int KIND, bool DEDUP, bool PERCELL, int SAMP, bool REC, bool COMPACT>
__global__ void __launch_bounds__(256, 2) tail_kernel(const ScenarioDev sc, const SimBuffers bf, const EpochArgs ep) {
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
    constexpr bool FAST = (SAMP == 0) && !REC;                // the fast round: exponential sampler, no event stream

    u32 lane;
    asm volatile("mov.u32 %0, %%laneid;" : "=r"(lane));                // opaque: kept in a register, not re-read per use
    // general path: event draws, one per lane: draw = F((X ^ lane_xor) + lane_add)
    const u64 lane_xor = lane == 0 ? NS_L_SPEC : lane == 1 ? NS_L_INDEX : lane == 2 ? NS_L_MIGR : NS_L_DISP;
    const u32 att_lane = lane >= 3u ? lane - 3u : 0u;                  // dispersal attempt of this lane within a pass
    const u64 att_add = (u64)att_lane * NS_GAMMA;
    // speculative round (SAMP 0): candidate and slot of this lane
    const u32 sp_c = lane >> 2, sp_q = lane & 3u;
    const u32 sp_dk = sp_c < NS_SPEC_NJ ? 0u : sp_c - NS_SPEC_NJ + 1u;
    const u64 sp_cand_add = (u64)(sp_c < NS_SPEC_NJ ? sp_c + 1u : 1u) * NS_GAMMA;
    const u64 sp_a_add = (KIND == 3 ? (u64)sp_q : 0ull) * NS_GAMMA;                       // slot A: attempt sp_q
    const u64 sp_b_xor = sp_q == 0 ? 0ull : sp_q == 1 ? NS_L_SPEC : sp_q == 2 ? NS_L_INDEX : NS_L_MIGR;   // slot B
    const bool sp_in_k = lane < 4u * NS_SPEC_NJ;
    const bool sp_add4 = sp_in_k && lane >= 4u, sp_add8 = sp_in_k && lane >= 8u, sp_add12 = sp_in_k && lane >= 12u, sp_add16 = sp_in_k && lane >= 16u;
    const u32 kmask = (1u << (4u * NS_SPEC_NJ)) - 1u;
    const u32 qb = lane & ~3u;
    unsigned long long c_events = 0, c_culled = 0, c_resamples = 0, c_exact = 0;   // warp-uniform
    u32 w_resamples = 0;                                                        // fast rounds: flushed into c_resamples per lineage
    // event-stream ring (REC): the warp reserves ep.rec_chunk (<= NS_REC_CHUNK) slots at a time, so that it waits for an atomic's return once per
    // chunk and not once per event; slots left over at the end get the sentinel key ~0, which sorts last and is dropped
    u32 rec_next = 0, rec_left = 0;
    auto record = [&](u32 r_loc, u32 r_k, u32 r_j, u64 r_f, u32 r_l2) {   // lane 0 only
        if (rec_left == 0u) { rec_next = atomicAdd(&bf.ctr->n_rec, ep.rec_chunk); rec_left = ep.rec_chunk; }
        const u32 ri = rec_next++; --rec_left;
        if (ri < bf.rec_cap) store_record(bf, ri, r_loc, r_k, r_j, r_f, r_l2);
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
        if (PERCELL) { uint2 cs = load_rate<SAMP>(sc, KIND == 3 ? xy_index(sc, cell) : cell); Cm = cs.x; sh = cs.y; }
        // lower bound of the search inside interval k: exact (f_last; -1 = fresh, none) for the general path, binary32 (fa_last)
        // for the fast round. After a fast round only fa_last is current (f_exact = false); the exact value is then the offset
        // of the last executed event (e_loc, k, e_j), recomputed when the general path needs it.
        i64 f_last = -1;
        bool f_exact = true;
        float fa_last = -1.0f, fm_last = 0.0f, ln2_over_mu = 0.0f, margin = 0.0f;   // fm_last: error margin of fa_last
        u32 e_loc = 0xFFFFFFFFu, e_j = 0, e_Cm = Cm, e_sh = sh;   // last executed event (origin, ordinal, rate of the origin's cell)
        if (FAST) { const float finv = rate_to_float(Cm, sh); ln2_over_mu = NS_LN2F * finv; margin = NS_MARGIN * (1.0f + finv); }
        const u32 cap_at = ep.max_steps ? ep.max_steps : 0xFFFFFFFFu;
        // pending duplicate check: the exchange of the last probing event (lane 0 holds its result)
        bool pend = false, p_T_known = true;
        u64 pold_lo = ~0ull, pold_hi = ~0ull;
        u32 p_lane = 0;                                    // the lane that issued the pending exchange and holds its result (warp-uniform)
        u32 p_loc = 0, p_k = 0, p_j = 0, p_l2 = 0;
        u64 p_T = 0;
        // consumes the pending exchange: true = this lineage is a duplicate at the pending event (culled, recorded)
        auto resolve_pending = [&]() -> bool {
            if (!DEDUP || !pend) return false;
            pend = false;
            const u32 ox = __shfl_sync(NS_FULL, (u32)pold_lo, (int)p_lane), oy = __shfl_sync(NS_FULL, (u32)(pold_lo >> 32), (int)p_lane);
            const u32 oz = __shfl_sync(NS_FULL, (u32)pold_hi, (int)p_lane), ow = __shfl_sync(NS_FULL, (u32)(pold_hi >> 32), (int)p_lane);
            if (ox == p_loc && oy == p_k && oz == p_j && ow != id) {   // another lineage executed it first (L687, L697)
                if (FAST && !p_T_known) { const uint2 pr = rate_of_loc<PERCELL>(sc, p_loc); p_T = exact_offset(ep.key, smt, p_loc, p_k, p_j, pr.x, pr.y); }
                if (lane == 0) {
                    bf.parent[id] = ow; bf.state[id] = 2;
                    bf.term_loc[id] = p_loc; bf.term_k[id] = p_k; bf.term_j[id] = p_j; bf.term_f[id] = p_T; bf.steps[id] = steps;
                }
                c_culled++;
                return true;
            }
            steps++;                                       // the pending event was really executed
            if (REC && lane == 0) record(p_loc, p_k, p_j, p_T, p_l2);
            return false;
        };

        for (;;) {   // one iteration = one search round (+ the event it finds)
            if (k == ep.k_stop) {   // epoch horizon: survivor (unless its last event turns out to be a duplicate)
                if (resolve_pending()) break;
                if (lane == 0) bf.q_out[atomicAdd(&bf.ctr->q_out, 1u)] = make_uint4(id, loc, cell, steps);
                break;
            }
            if (FAST) {
                // ---- fast rounds: the search in binary32 with a margin (see approx_exp_time), every candidate's outcome from its own four
                // lanes. The loop commits clean events (99 %: candidate in the set, unambiguous comparisons, an attempt accepted, no
                // speciation, no duplicate, no step cap) and leaves at the first round that is not, which the general code below redoes.
                // A duplicate check still pending from the general code is settled first (rare: the loop is entered once per ~40 events and
                // one event in eight probes). Inside the loop the pending event is then always the last committed one, (e_loc, k, e_j), its
                // result sits in lane p_lane, and the step count includes it (steps_all; `steps` counts confirmed events only).
                if (DEDUP && pend) { if (resolve_pending()) break; }
                u32 steps_all = steps;
                bool lpend = false;
                // s = the stream state of this lane's candidate interval, prime(loc, k + sp_dk). Inside the loop the NEXT round's states are
                // primed ahead of the vote: every candidate's four lanes prime the four intervals the next round looks at from the
                // candidate's own outcome (its target location, its interval + 0..3), while the ballots pick the winner; after the vote the
                // states come from the winner's lanes by shuffle instead of six Feistel rounds at the head of the next round's chain.
                u64 s = prime(ep.key, loc, k + sp_dk);
                // continuation rounds: when none of the five points of interval k looked at lies after the bound and the interval is not
                // exhausted either (1.1 % of the events: a late bound in a new stream with many early points), the next round looks at the
                // following five points, j0 + 1 .. j0 + 5, with the partial sum a0 carried over, instead of falling back to the exact path
                u32 j0 = 0;
                float a0 = 0.0f;
                u64 cand_add = sp_cand_add;
                // attempt round (after the loop): the event is known and everything about it is settled except its dispersal: the first four
                // attempts were all rejected (1.4 % of the events of C5's tail: lineages in sparsely inhabited neighbourhoods), or a target at
                // or before the first accepted attempt fell into a crowded bucket of the rounded-normal guide (0.2 %)
                bool rs = false, rs_rej = false;   // rs_rej: four determined attempts, all rejected -> attempts 4..35 with the fast lookup
                u32 rs_k2 = 0, rs_j2 = 0, rs_xlo = 0, rs_xhi = 0;
                u64 rs_X = 0;
                float rs_a = 0.0f;
                for (;;) {
                    const u64 X = s + cand_add;
                    u64 ua, ub;
                    hashF2((X ^ NS_L_DISP) + sp_a_add, X ^ sp_b_xor, ua, ub);
                    // duplicate check of the candidate, decided per lane ahead of the selection: whether its event probes the cache, and where.
                    // The winner's first lane issues the exchange itself and keeps the result (no shuffle of X, no hash after the vote).
                    const u32 ch = DEDUP ? cache_hash(X) : 0u;
                    const u32 prm = DEDUP ? __ballot_sync(NS_FULL, cache_probes(ch, ep.probe_mask)) : 0u;
                    const u32 ubh = (u32)(ub >> 32);
                    ua |= (u64)(ubh & ep.zero);       // keeps the two evaluations interleaved (slot A's chain is the longer one and would go first)
                    const u32 bm = __ballot_sync(NS_FULL, bern(ub, sp_q == 3u ? ep.thr_m : ep.thr_nu));   // bit 4c+1: speciation, 4c+3: migration
                    const u32 xi_lo = __shfl_sync(NS_FULL, (u32)ub, (int)(qb + 2u)), xi_hi = __shfl_sync(NS_FULL, ubh, (int)(qb + 2u));
                    u32 loc2o, c2o, tie; uint2 cso = make_uint2(Cm, sh); bool acc, bad;
                    fast_slot_a<KIND, PERCELL, COMPACT>(sc, gl, sp_q, lane, bm, cell, k + sp_dk, ua, xi_lo, xi_hi, loc2o, c2o, cso, acc, bad, tie);
                    // slot B of the lanes with sp_q == 0: approximate offsets of the candidates (partial sums over the points of interval k)
                    // (the draw is tied to the target cell of slot A by an OR with zero: the table gathers, which have the longest latency,
                    // are then issued before this chain starts)
                    float a = sp_q == 0u ? approx_exp_time(ubh | (c2o & ep.zero), ln2_over_mu) : 0.0f;
                    if (lane == 0) a += a0;
                    // (the partial sums are tied to the gathered table entry by an OR with zero: ptxas otherwise places the gather, whose
                    // consumers come late, behind the whole shuffle / compare / ballot chain, and its latency ends up on the lineage's chain
                    // instead of under it. With the tie the gather is issued first and the logarithms run while it is in flight.)
                    {   // five partial sums in two shuffle levels: a_j + a_{j-1} + a_{j-2}, then + the same sum three candidates below
                        // (one level with four shuffles and an add tree measured slower: 0.467 against 0.463 us)
                        const float y1 = __shfl_up_sync(NS_FULL, a, 4), y2 = __shfl_up_sync(NS_FULL, a, 8);
                        float b3 = a;
                        if (sp_add4) b3 += y1;
                        if (sp_add8) b3 += y2;
                        const float y3 = __shfl_up_sync(NS_FULL, b3, 12);
                        a = b3;
                        if (sp_add12) a += y3;
                    }
                    if (COMPACT) a = __uint_as_float(__float_as_uint(a) | (tie & ep.zero));
                    const float mc = margin + fm_last;
                    const bool ins = a < 1.0f - margin, outs = a > 1.0f + margin;
                    bool aft = a > fa_last + mc, bef = a < fa_last - mc;
                    // a lineage that stayed where it was (self-dispersal) sees the points of the same stream again: after the last event
                    // means a larger ordinal, exactly (the partial sums are the same numbers as in the round before)
                    if (loc == e_loc && fa_last >= 0.0f) { aft = j0 + sp_c + 1u > e_j; bef = !aft; }
                    const bool kvalid = (ep.k_stop - k) > sp_dk;              // never look at or past the horizon (k < k_stop here)
                    // draws with hi < 2^20 (coarse logarithm) or hi >= 2^32 - 2^8 (an increment that may round to zero) are not decided here
                    const bool amb = (ubh - (1u << 20) >= 0xFFEFFF00u) || !(ins || outs) || (sp_in_k && !(aft || bef));
                    const u32 evm = __ballot_sync(NS_FULL, sp_q == 0u && ins && (sp_in_k ? aft : kvalid));
                    const u32 crm = __ballot_sync(NS_FULL, sp_q == 0u && outs);
                    const u32 okm = __ballot_sync(NS_FULL, acc);
                    // trouble: an ambiguous comparison anywhere, or (the lane that holds the result of the pending exchange) a match there:
                    // another lineage executed the pending event first and this one is a duplicate
                    bool culled = false;
                    if (DEDUP) culled = lane == p_lane && lpend && (u32)pold_lo == e_loc && (u32)(pold_lo >> 32) == k && (u32)pold_hi == e_j && (u32)(pold_hi >> 32) != id;
                    const u32 trm = __ballot_sync(NS_FULL, (sp_q == 0u && amb) || culled);
                    const u32 badm = KIND == 3 ? __ballot_sync(NS_FULL, bad) : 0u;
                    // every candidate's outcome: the first accepted attempt of its four lanes (the sequential algorithm's choice, R16)
                    const int qsrc = (int)(qb + ((u32)first_bit(((okm >> qb) & 15u) | 16u) & 3u));
                    const u32 loc2q = __shfl_sync(NS_FULL, loc2o, qsrc), cq = __shfl_sync(NS_FULL, c2o, qsrc);
                    u32 Cmq = Cm, shq = sh;
                    if (PERCELL) { Cmq = __shfl_sync(NS_FULL, cso.x, qsrc); shq = __shfl_sync(NS_FULL, cso.y, qsrc); }
                    const u64 s_own = prime(ep.key, loc2q, k + sp_dk + sp_q);    // next round's state of interval (this candidate's) + sp_q, if it wins
                    // the winner: first point of interval k after fa_last, else (interval exhausted, L719, L727) the first non-empty later interval
                    const u32 m0 = evm & kmask;
                    const u32 m1 = (crm & kmask) ? (evm & ~kmask) : 0u;
                    const u32 wm = m0 ? m0 : m1;
                    const u32 wl = (u32)first_bit(wm | 0x80000000u);
                    const u32 q4 = 15u << wl;
                    const u32 spec_w = (KIND == 1 && cell == 0) ? 0u : ((bm >> wl) & 2u);
                    const u32 steps_e = steps_all + 1u;                 // step count after this event
                    // clean: a winner, no trouble at the time lanes or in the winner's lanes, an attempt accepted, no speciation, no step cap
                    // (an undetermined target matters only up to the winner's first accepted attempt -- later attempts are never looked at:
                    // x ^ (x - 1) = the bits up to and including the lowest set bit of x)
                    const u32 okw = okm & q4;
                    const bool clean = wm != 0u && ((trm & 0x11111111u) | (badm & q4 & (okw ^ (okw - 1u))) | spec_w) == 0u && okw != 0u && steps_e < cap_at;
                    if (!clean) {                      // warp-uniform: every term comes out of a ballot or is lineage state
                        if (wm == 0u && (crm & kmask) == 0u && (trm & 0x11111111u) == 0u && j0 < 25u) {   // continuation round (see above)
                            a0 = __shfl_sync(NS_FULL, a, (int)(4u * (NS_SPEC_NJ - 1u)));
                            j0 += NS_SPEC_NJ;
                            if (sp_in_k) cand_add += (u64)NS_SPEC_NJ * NS_GAMMA;
                            continue;
                        }
                        // (here with a winner, no ambiguity, no duplicate, no speciation: what is wrong is the winner's dispersal -- four
                        // attempts rejected, or an undetermined target at or before the first accepted one)
                        if (KIND == 3 && wm != 0u && ((trm & 0x11111111u) | spec_w) == 0u && steps_e < cap_at) {
                            const u32 wc = wl >> 2;
                            rs = true; rs_rej = okw == 0u && (badm & q4) == 0u;
                            rs_k2 = k + (wc < NS_SPEC_NJ ? 0u : wc - NS_SPEC_NJ + 1u); rs_j2 = wc < NS_SPEC_NJ ? j0 + wc + 1u : 1u;
                            rs_X = __shfl_sync(NS_FULL, X, (int)wl); rs_a = __shfl_sync(NS_FULL, a, (int)wl);
                            rs_xlo = __shfl_sync(NS_FULL, (u32)ub, (int)(wl + 2u)); rs_xhi = __shfl_sync(NS_FULL, ubh, (int)(wl + 2u));
                        }
                        break;
                    }
                    // commit: event (loc, k2, j2) executed, the lineage moves to the winner's target
                    const u32 wc = wl >> 2;
                    const u32 k2 = k + (wc < NS_SPEC_NJ ? 0u : wc - NS_SPEC_NJ + 1u);
                    const u32 j2 = wc < NS_SPEC_NJ ? j0 + wc + 1u : 1u;
                    const u32 loc2 = __shfl_sync(NS_FULL, loc2q, (int)wl), cell2 = __shfl_sync(NS_FULL, cq, (int)wl);
                    const float a_w = __shfl_sync(NS_FULL, a, (int)wl);
                    if (KIND == 3) w_resamples += (u32)first_bit((okm >> wl) & 15u);
                    steps_all = steps_e;
                    if (DEDUP) {                                       // (a clean round has confirmed the event that was pending)
                        lpend = (prm >> wl) & 1u;
                        atomic_exch_128_if(lpend && lane == wl, &bf.cache[ch & bf.cache_mask], make_uint4(loc, k2, j2, id), pold_lo, pold_hi);
                        if (lpend) p_lane = wl;
                    }
                    e_loc = loc; e_j = j2; e_Cm = Cm; e_sh = sh; f_exact = false; fa_last = a_w; fm_last = margin;
                    if (PERCELL) {
                        Cm = __shfl_sync(NS_FULL, Cmq, (int)wl); sh = __shfl_sync(NS_FULL, shq, (int)wl);
                        const float finv = rate_to_float(Cm, sh);
                        ln2_over_mu = NS_LN2F * finv; margin = NS_MARGIN * (1.0f + finv);
                    }
                    k = k2; loc = loc2; cell = cell2;
                    s = __shfl_sync(NS_FULL, s_own, (int)(wl + sp_dk));
                    if (j0) { j0 = 0; a0 = 0.0f; cand_add = sp_cand_add; }
                }
                steps = steps_all;
                if (DEDUP && lpend) {          // hand the pending check over to the general code, which keeps the result in lane 0
                    steps = steps_all - 1u; pend = true; p_loc = e_loc; p_k = k; p_j = e_j; p_T_known = false;
                    pold_lo = __shfl_sync(NS_FULL, pold_lo, (int)p_lane); pold_hi = __shfl_sync(NS_FULL, pold_hi, (int)p_lane);
                }
                p_lane = 0u;
                if (KIND == 3 && rs) {
                    // the 32 lanes evaluate attempts 0 .. 31 of the event (loc, rs_k2, rs_j2) with the exact rounded-normal lookup: one hash,
                    // the lookups and the gather, instead of the exact path. (The pending duplicate check, if any, was clear in the round
                    // that found the event: it is resolved first.)
                    u32 c2b, loc2b, okb, fa, nres;
                    uint2 csb = make_uint2(Cm, sh);
                    if (rs_rej) {
                        const u64 ua2 = hashF((rs_X ^ NS_L_DISP) + (u64)(4u + lane) * NS_GAMMA);
                        u32 tieb; bool accb, badb;
                        fast_slot_a<KIND, PERCELL, COMPACT>(sc, gl, 0u, lane, 0u, cell, rs_k2, ua2, rs_xlo, rs_xhi, loc2b, c2b, csb, accb, badb, tieb);
                        okb = __ballot_sync(NS_FULL, accb);
                        const u32 bdb = __ballot_sync(NS_FULL, badb);
                        fa = (u32)first_bit(okb | 0x80000000u);
                        if (bdb & ((2u << fa) - 1u)) okb = 0u;          // an undetermined target at or before the first accepted: exact path
                        nres = 4u + fa;
                    } else {
                        const u64 ua2 = hashF((rs_X ^ NS_L_DISP) + (u64)lane * NS_GAMMA);
                        u32 db, pfb; bool badb;
                        gauss_target<PERCELL, SAMP, COMPACT, false>(sc, gl, cell & 0xFFFFu, cell >> 16, ua2, rs_k2, c2b, db, pfb, csb, badb);
                        loc2b = pfb + ((db == 1u) ? 0u : mulhi64_u32_parts(rs_xlo, rs_xhi, db));
                        okb = __ballot_sync(NS_FULL, db > 0u);
                        fa = (u32)first_bit(okb | 0x80000000u);
                        nres = fa;
                    }
                    if (okb != 0u) {
                        if (resolve_pending()) break;
                        bool probes = false;
                        if (DEDUP) {
                            const u32 h = cache_hash(rs_X);
                            probes = cache_probes(h, ep.probe_mask);
                            atomic_exch_128_if(probes && lane == 0, &bf.cache[h & bf.cache_mask], make_uint4(loc, rs_k2, rs_j2, id), pold_lo, pold_hi);
                            if (probes) { p_loc = loc; p_k = rs_k2; p_j = rs_j2; p_T_known = false; pend = true; }
                        }
                        if (!probes) steps++;
                        w_resamples += nres;
                        e_loc = loc; e_j = rs_j2; e_Cm = Cm; e_sh = sh; f_exact = false; fa_last = rs_a; fm_last = margin;
                        if (PERCELL) {
                            Cm = __shfl_sync(NS_FULL, csb.x, (int)fa); sh = __shfl_sync(NS_FULL, csb.y, (int)fa);
                            const float finv = rate_to_float(Cm, sh);
                            ln2_over_mu = NS_LN2F * finv; margin = NS_MARGIN * (1.0f + finv);
                        }
                        k = rs_k2; loc = __shfl_sync(NS_FULL, loc2b, (int)fa); cell = __shfl_sync(NS_FULL, c2b, (int)fa);
                        continue;
                    }
                }
                // the round that was not clean is done below in exact arithmetic, from the exact lower bound
                if (!f_exact) { f_last = (i64)exact_offset(ep.key, smt, e_loc, k, e_j, e_Cm, e_sh); f_exact = true; }
                c_exact++;
            }
            u32 j;
            u64 Te, Xe;
            // outcome of the event when the speculative round evaluated it already
            bool have = false, h_spec = false;
            u32 h_loc2 = 0, h_cell2 = 0, h_Cm2 = Cm, h_sh2 = sh;
            if (SAMP == 1) {
                // S1 (Poisson sampler, Cm = thinning threshold of the cell)
                if (!tail_search_poisson<PERCELL>(ep.key, smt, lane, loc, k, f_last, ep.k_stop, Cm, j, Te, Xe)) continue;
            } else {
                // ---- S1 + S2 + S3 side by side: 8 candidate events x (4 attempts | time, speciation, index, migration) -----------
                const bool kvalid = (ep.k_stop - k) > sp_dk;              // never look at or past the horizon (k < k_stop here)
                const u64 X = prime(ep.key, loc, k + sp_dk) + sp_cand_add;
                u64 ua, ub;
                hashF2((X ^ NS_L_DISP) + sp_a_add, X ^ sp_b_xor, ua, ub);
                const u32 bm = __ballot_sync(NS_FULL, bern(ub, sp_q == 3u ? ep.thr_m : ep.thr_nu));   // bit 4c+1: speciation, 4c+3: migration
                // slot A: dispersal target (gathers in flight during the arithmetic below)
                u32 c2 = 0, d = 0, pf = 0;
                uint2 cs = make_uint2(Cm, sh);
                bool bad = false;
                if (KIND == 0) {
                    if (sp_q == 0u) { pf = mulhi64_u32(ua, (u32)sc.n_locations); d = 1u; }
                } else if (KIND == 1) {
                    if (sp_q == 0u) {
                        const bool to_meta = (cell != 0) || ((bm >> (lane + 3u)) & 1u);
                        if (to_meta) { pf = sc.J_local + mulhi64_u32(ua, sc.J_meta); c2 = 1u; }
                        else pf = mulhi64_u32(ua, sc.J_local);
                        d = 1u;
                    }
                } else if (KIND == 2) {
                    if (sp_q == 0u) {
                        const u32 n = sc.ncells, col = __umulhi((u32)(ua >> 32), n);
                        const uint2 e = __ldg(&sc.alias[(size_t)cell * n + col]);
                        c2 = ((u32)ua < e.x) ? col : e.y;
                        pf = ldg_u32_ordered(&sc.prefix[c2]);
                        if (PERCELL) cs = ldg_v2_ordered(&sc.scale[c2]);
                        d = ldg_u8_ordered(&sc.hab8[c2]);
                        if (d == 255u) d = __ldg(&sc.deme32[c2]);
                    }
                } else {
                    gauss_target<PERCELL, SAMP, COMPACT, true>(sc, gl, cell & 0xFFFFu, cell >> 16, ua, k + sp_dk, c2, d, pf, cs, bad);
                }
                // the outcome of EVERY candidate from its own four lanes, before the search says which one it is: first accepted
                // attempt (= the sequential algorithm's choice, R16), its cell and prefix, the index draw of the candidate
                const u32 okm = __ballot_sync(NS_FULL, d > 0u);
                const u32 badm = KIND == 3 ? __ballot_sync(NS_FULL, bad) : 0u;
                const int qsrc = (int)(qb + ((u32)first_bit(((okm >> qb) & 15u) | 16u) & 3u));
                const u32 dq = __shfl_sync(NS_FULL, d, qsrc), pq = __shfl_sync(NS_FULL, pf, qsrc), cq = __shfl_sync(NS_FULL, c2, qsrc);
                u32 Cmq = Cm, shq = sh;
                if (PERCELL) { Cmq = __shfl_sync(NS_FULL, cs.x, qsrc); shq = __shfl_sync(NS_FULL, cs.y, qsrc); }
                const u64 xiq = __shfl_sync(NS_FULL, ub, (int)(qb + 2u));
                const u32 loc2q = pq + ((dq == 1u) ? 0u : mulhi64_u32(xiq, dq));

                // slot B of the lanes with sp_q == 0: the time draw of the candidate (every lane runs the arithmetic)
                const u64 T1 = scale_exp(neglog(ub, smt), Cm, sh);
                // partial sums T_j over the points of interval k: lanes 0, 4, .., 16 (offsets of 1, 2, 4 candidates)
                u64 T = sp_q == 0u ? T1 : 0ull;
                { const u64 y = __shfl_up_sync(NS_FULL, T, 4); if (sp_add4) T += y; }
                { const u64 y = __shfl_up_sync(NS_FULL, T, 8); if (sp_add8) T += y; }
                { const u64 y = __shfl_up_sync(NS_FULL, T, 16); if (sp_add16) T += y; }
                const bool inside = T < NS_TWO48;
                const u32 evm = __ballot_sync(NS_FULL, sp_q == 0u && inside && (sp_in_k ? ((i64)T > f_last) : kvalid));
                const u32 crm = __ballot_sync(NS_FULL, sp_q == 0u && !inside);
                const u32 m0 = evm & kmask;                    // next event is in interval k
                const u32 m1 = (crm & kmask) ? (evm & ~kmask) : 0u;   // interval k exhausted (L719, L727): first non-empty interval after it
                const u32 wm = m0 ? m0 : m1;
                if (wm) {
                    const int wl = first_bit(wm);              // lane of the winning candidate's slot-A attempt 0 / time draw
                    const u32 wc = (u32)wl >> 2;
                    k += wc < NS_SPEC_NJ ? 0u : wc - NS_SPEC_NJ + 1u;
                    j = wc < NS_SPEC_NJ ? wc + 1u : 1u;
                    Te = __shfl_sync(NS_FULL, T, wl); Xe = __shfl_sync(NS_FULL, X, wl);
                    h_spec = !(KIND == 1 && cell == 0) && ((bm >> ((u32)wl + 1u)) & 1u);
                    const u32 acc = (okm >> (u32)wl) & 15u;
                    if (h_spec) have = true;
                    else if (acc && !((badm >> (u32)wl) & 15u)) {
                        h_loc2 = __shfl_sync(NS_FULL, loc2q, wl); h_cell2 = __shfl_sync(NS_FULL, cq, wl);
                        if (PERCELL) { h_Cm2 = __shfl_sync(NS_FULL, Cmq, wl); h_sh2 = __shfl_sync(NS_FULL, shq, wl); }
                        if (KIND == 3) c_resamples += (u32)first_bit(acc);
                        have = true;
                    }
                } else if (crm & kmask) {                      // all speculated intervals empty / beyond the horizon
                    const u32 gap = ep.k_stop - 1u - k;
                    k = k + 1u + (gap < NS_SPEC_ND ? gap : NS_SPEC_ND); f_last = -1; fa_last = -1.0f; fm_last = 0.0f;
                    continue;
                } else {
                    // more than NS_SPEC_NJ points of interval k at or before f_last: continue the scan one draw at a time
                    u64 Tc = __shfl_sync(NS_FULL, T, 4 * (NS_SPEC_NJ - 1u)), Xc = __shfl_sync(NS_FULL, X, 4 * (NS_SPEC_NJ - 1u));
                    u32 jc = NS_SPEC_NJ;
                    bool found = false;
                    for (;;) {
                        jc += 1u; Xc += NS_GAMMA;
                        Tc += scale_exp(neglog(draw_time(Xc), smt), Cm, sh);
                        if (Tc >= NS_TWO48) break;
                        if ((i64)Tc > f_last) { found = true; break; }
                    }
                    if (!found) { k += 1u; f_last = -1; fa_last = -1.0f; fm_last = 0.0f; continue; }
                    j = jc; Te = Tc; Xe = Xc;
                }
            }

            // ---- event (loc, k, j) at offset Te --------------------------------------------------------------
            // S5: the previous probing event's exchange is consumed before this event may publish a cache entry
            if (resolve_pending()) break;
            bool probes = false;
            if (DEDUP) {
                const u32 h = cache_hash(Xe);
                probes = cache_probes(h, ep.probe_mask);
                atomic_exch_128_if(probes && lane == 0, &bf.cache[h & bf.cache_mask], make_uint4(loc, k, j, id), pold_lo, pold_hi);
                if (probes) { p_loc = loc; p_k = k; p_j = j; p_T = Te; p_T_known = true; pend = true; }
            }
            if (!probes) steps++;
            bool speciates = h_spec;
            u32 loc2 = h_loc2, cell2 = h_cell2, Cm2 = h_Cm2, sh2 = h_sh2;
            bool ok = true;
            if (!have) {
                // S2 + S3, general path: all draws of the event in one hash evaluation across the lanes
                const u64 xb = Xe ^ lane_xor;
                u64 u = hashF(xb + att_add);
                const bool can_speciate = !(KIND == 1 && cell == 0);      // local community of the implicit model: nu = 0 (L1830)
                const u32 bm = __ballot_sync(NS_FULL, bern(u, lane == 2 ? ep.thr_m : ep.thr_nu));
                speciates = can_speciate && (bm & 1u);
                loc2 = loc; cell2 = cell; Cm2 = Cm; sh2 = sh;
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
                            bool bad_;
                            if (lane >= 3u) gauss_target<PERCELL, SAMP, COMPACT, false>(sc, gl, x0, y0, u, k, c2, d, pf, cs, bad_);   // attempt r0 + lane - 3 (R16: redraw the whole (dx, dy) pair)
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
            if (FAST) { e_loc = loc; e_j = j; e_Cm = Cm; e_sh = sh; }
            f_last = (i64)Te; loc = loc2; cell = cell2; Cm = Cm2; sh = sh2;
            if (FAST) {
                f_exact = true; fa_last = (float)Te * 0x1p-48f; fm_last = 2.4e-07f;   // binary32 rounding of an offset < 1
                if (PERCELL) { const float finv = rate_to_float(Cm, sh); ln2_over_mu = NS_LN2F * finv; margin = NS_MARGIN * (1.0f + finv); }
            }
        }
        c_events += steps - qe.w;                  // events this lineage executed in this launch
        c_resamples += w_resamples; w_resamples = 0;
    }
    if (REC) {   // sentinels into the reserved slots that stayed empty
        const u32 nx = __shfl_sync(NS_FULL, rec_next, 0), lf = __shfl_sync(NS_FULL, rec_left, 0);
        for (u32 q = lane; q < lf; q += 32u) {
            const u32 ri = nx + q;
            if (ri < bf.rec_cap) store_sentinel(bf, ri);          // sentinel: sorts last, dropped
        }
    }
    if (lane == 0) {
        if (c_events) atomicAdd((unsigned long long *)&bf.ctr->n_events, c_events);
        if (c_culled) atomicAdd((unsigned long long *)&bf.ctr->n_culled, c_culled);
        if (c_resamples) atomicAdd((unsigned long long *)&bf.ctr->resamples, c_resamples);
        if (c_exact) atomicAdd((unsigned long long *)&bf.ctr->tail_rounds_exact, c_exact);
    }
}

}  // namespace necsim
