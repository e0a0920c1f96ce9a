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
//   - every lane also evaluates the speciation draw and the first dispersal attempt of ITS candidate (with the
//     habitat / prefix / turnover-scale gathers) while its -ln chain is in flight, so that when the winning
//     candidate is known the event is already decided and the next search starts at once;
//   - the duplicate-culling exchange of an event is issued when the event is selected and consumed one event
//     later (never after another cache insertion: an unconfirmed lineage must not publish entries);
//   - rejected dispersal targets fall back to eight attempts at a time.
#pragma once
#include "sim_kernel.cuh"

namespace necsim {

#define NS_TAIL_ATTEMPTS 8u

// Dispersal of one candidate event (stream position X), written branch-free so that it schedules into the
// latency of the candidate's -ln chain. KIND 0..2: the complete dispersal. KIND 3: attempt 0 only;
// ok = target is habitat; exact = false where the table lookups need their rare exact path (then the caller
// re-evaluates from attempt 0).
template <int KIND, bool PERCELL>
__device__ __forceinline__ void candidate_disperse(const ScenarioDev &sc, u64 thr_m, u64 X, u32 cell, const GaussLut &gl,
                                                   u32 &loc2, u32 &cell2, u32 &Cm2, u32 &sh2, bool &ok, bool &exact) {
    ok = true; exact = true;
    u32 idx2 = 0;
    if (KIND == 0) {
        loc2 = mulhi64_u32(draw_disp(X, 0), (u32)sc.n_locations); cell2 = 0;
    } else if (KIND == 1) {
        const u64 x = draw_disp(X, 0);
        const bool to_meta = (cell != 0) || bern(draw_migr(X), thr_m);
        const u32 lm = sc.J_local + mulhi64_u32(x, sc.J_meta), ll = mulhi64_u32(x, sc.J_local);
        loc2 = to_meta ? lm : ll; cell2 = to_meta ? 1u : 0u;
    } else if (KIND == 2) {
        const u64 x = draw_disp(X, 0);
        const u32 n = sc.ncells, col = __umulhi((u32)(x >> 32), n);
        const uint2 e = __ldg(&sc.alias[(size_t)cell * n + col]);
        cell2 = ((u32)x < e.x) ? col : e.y;
        const u32 d = __ldg(&sc.hab8[cell2]);
        exact = d != 255u;
        loc2 = __ldg(&sc.prefix[cell2]) + mulhi64_u32(draw_index(X), d);     // d = 1 gives index 0
        idx2 = cell2;
    } else {
        const u64 x = draw_disp(X, 0);
        bool e1, e2;
        const u32 xx = wrap_add(cell & 0xFFFFu, gauss_disp_fast(gl, (u32)(x >> 32), e1), sc.width);
        const u32 yy = wrap_add(cell >> 16, gauss_disp_fast(gl, (u32)x, e2), sc.height);
        idx2 = yy * sc.width + xx;
        cell2 = (yy << 16) | xx;
        const u32 d = __ldg(&sc.hab8[idx2]);
        ok = d > 0u; exact = e1 && e2 && d != 255u;
        loc2 = __ldg(&sc.prefix[idx2]) + mulhi64_u32(draw_index(X), d);
    }
    if (PERCELL) { const uint2 cs = __ldg(&sc.scale[idx2]); Cm2 = cs.x; sh2 = cs.y; }
}

template <int KIND, bool DEDUP, bool PERCELL>
__global__ void __launch_bounds__(256) tail_kernel(const ScenarioDev sc, const SimBuffers bf, const EpochArgs ep) {
    __shared__ unsigned short sQ[512];
    __shared__ u64 sA[512];
    __shared__ u32 sG[KIND == 3 ? 1024 : 1];
    __shared__ uint2 sG2[KIND == 3 ? NS_G2_LEN : 1];
    for (u32 i = threadIdx.x; i < 512; i += blockDim.x) { sQ[i] = NEGLOG_Q_DEV[i]; sA[i] = NEGLOG_A_DEV[i]; }
    if (KIND == 3) gauss_stage(sc, sG, sG2);
    __syncthreads();
    GaussLut gl; gl.tg = sG; gl.g2 = sG2; gl.R = sc.R;

    const u32 lane = threadIdx.x & 31u, half = lane >> 4, sub = lane & 15u;
    const u32 jj = half ? 1u : sub + 1u;                               // ordinal of this lane's candidate
    unsigned long long c_events = 0, c_culled = 0, c_resamples = 0;   // warp-uniform

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
        if (PERCELL) { uint2 cs = __ldg(&sc.scale[KIND == 3 ? xy_index(sc, cell) : cell]); Cm = cs.x; sh = cs.y; }
        // pending duplicate check: the exchange of the last probing event (lane 0 holds its result)
        bool pend = false;
        uint4 pold = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
        u32 p_loc = 0, p_k = 0, p_j = 0;
        u64 p_T = 0;
        // consumes the pending exchange: true = this lineage is a duplicate at the pending event (culled, recorded)
        auto resolve_pending = [&]() -> bool {
            if (!DEDUP || !pend) return false;
            pend = false;
            const u32 ox = __shfl_sync(NS_FULL, pold.x, 0), oy = __shfl_sync(NS_FULL, pold.y, 0);
            const u32 oz = __shfl_sync(NS_FULL, pold.z, 0), ow = __shfl_sync(NS_FULL, pold.w, 0);
            if (ox == p_loc && oy == p_k && oz == p_j && ow != id) {   // another lineage executed it first (L687, L697)
                if (lane == 0) {
                    bf.parent[id] = ow; bf.state[id] = 2;
                    bf.term_loc[id] = p_loc; bf.term_k[id] = p_k; bf.term_j[id] = p_j; bf.term_f[id] = p_T; bf.steps[id] = steps;
                }
                c_culled++;
                return true;
            }
            steps++; c_events++;                                       // the pending event was really executed
            return false;
        };

        for (;;) {   // one iteration = one search round (+ the event it finds)
            if (k == ep.k_stop) {   // epoch horizon: survivor (unless its last event turns out to be a duplicate)
                if (resolve_pending()) break;
                if (lane == 0) bf.q_out[atomicAdd(&bf.ctr->q_out, 1u)] = make_uint4(id, loc, cell, steps);
                break;
            }
            const bool can_speciate = !(KIND == 1 && cell == 0);      // local community of the implicit model: nu = 0 (L1830)
            // ---- S1-S3 for this lane's candidate event, speculatively: time, speciation and dispersal draws --------
            const u64 kk64 = (u64)k + (half ? (u64)(1u + sub) : 0ull);
            const bool kvalid = kk64 < (u64)ep.k_stop;                // never look at or past the horizon
            u64 X = prime(ep.key, loc, (u32)kk64) + (u64)jj * NS_GAMMA;
            const u64 T1 = scale_exp(neglog(draw_time(X), sQ, sA), Cm, sh);
            bool e_spec = can_speciate && bern(draw_spec(X), ep.thr_nu);
            u32 e_loc2 = loc, e_cell2 = cell, e_Cm = Cm, e_sh = sh;
            bool e_ok, e_exact;
            candidate_disperse<KIND, PERCELL>(sc, ep.thr_m, X, cell, gl, e_loc2, e_cell2, e_Cm, e_sh, e_ok, e_exact);
            // partial sums over each 16-lane half (half 1 keeps its single draws: first points of fresh intervals)
            u64 T = T1;
#pragma unroll
            for (int o = 1; o < 16; o <<= 1) {
                const u64 t = __shfl_up_sync(NS_FULL, T, o, 16);
                if ((int)sub >= o) T += t;
            }
            if (half) T = T1;
            const bool inside = T < NS_TWO48;
            const u32 evm = __ballot_sync(NS_FULL, inside && (half ? kvalid : ((i64)T > f_last)));
            const u32 crm = __ballot_sync(NS_FULL, !inside);
            u32 j;
            int src;
            if (evm & 0xFFFFu) {                       // next event is in interval k
                src = __ffs(evm & 0xFFFFu) - 1;
                j = (u32)src + 1u;
            } else if (crm & 0xFFFFu) {                // interval k exhausted (L719, L727): first non-empty interval after it
                const u32 gap = ep.k_stop - 1u - k;    // k < k_stop here
                const u32 nvalid = gap < 16u ? gap : 16u;
                const u32 hm = evm >> 16;
                if (!hm) { k = k + 1u + nvalid; f_last = -1; continue; }   // all speculated intervals empty / beyond the horizon
                src = 16 + __ffs(hm) - 1;
                k = k + 1u + (u32)(src - 16); j = 1u;
            } else {
                // more than 16 points of interval k at or before f_last (large mu): continue the scan one draw at a time
                u64 Tc = __shfl_sync(NS_FULL, T, 15), Xc = __shfl_sync(NS_FULL, X, 15);
                u32 jc = 16u;
                bool found = false;
                for (;;) {
                    jc += 1u; Xc += NS_GAMMA;
                    Tc += scale_exp(neglog(draw_time(Xc), sQ, sA), Cm, sh);
                    if (Tc >= NS_TWO48) break;
                    if ((i64)Tc > f_last) { found = true; break; }
                }
                if (!found) { k += 1u; f_last = -1; continue; }
                // every lane evaluates the same candidate: lane 0 serves as the source below
                j = jc; T = Tc; X = Xc; src = 0;
                e_spec = can_speciate && bern(draw_spec(X), ep.thr_nu);
                e_loc2 = loc; e_cell2 = cell; e_Cm = Cm; e_sh = sh;
                candidate_disperse<KIND, PERCELL>(sc, ep.thr_m, X, cell, gl, e_loc2, e_cell2, e_Cm, e_sh, e_ok, e_exact);
            }
            const u64 Te = __shfl_sync(NS_FULL, T, src);
            const u32 flags = __shfl_sync(NS_FULL, (e_spec ? 1u : 0u) | (e_ok ? 2u : 0u) | (e_exact ? 4u : 0u), src);
            u32 loc2 = __shfl_sync(NS_FULL, e_loc2, src), cell2 = __shfl_sync(NS_FULL, e_cell2, src);
            u32 Cm2 = Cm, sh2 = sh;
            if (PERCELL) { Cm2 = __shfl_sync(NS_FULL, e_Cm, src); sh2 = __shfl_sync(NS_FULL, e_sh, src); }
            const bool speciates = flags & 1u;
            bool ok = (flags & 6u) == 6u;              // accepted by the fast path

            // ---- event (loc, k, j) at offset Te --------------------------------------------------------------
            // S5: the previous probing event's exchange is consumed before this event may publish a cache entry
            if (resolve_pending()) break;
            bool probes = false;
            if (DEDUP) {
                const u32 h = cache_hash(loc, k, j);
                probes = cache_probes(h, ep.probe_mask);
                if (probes) {
                    if (lane == 0) pold = atomic_exch_128(&bf.cache[h & bf.cache_mask], make_uint4(loc, k, j, id));
                    p_loc = loc; p_k = k; p_j = j; p_T = Te; pend = true;
                }
            }
            if (!probes) { steps++; c_events++; }
            if (KIND >= 2 && !speciates && !ok) {
                // S3 slow path: exact lookups; attempts r0.. eight at a time (R16). Attempt 0 is known rejected when
                // the fast path was exact.
                const u64 Xe = __shfl_sync(NS_FULL, X, src);
                if (KIND == 2) {
                    u32 rs = 0;
                    ok = disperse<2>(sc, ep.thr_m, Xe, cell, loc2, cell2, gl, rs);
                    if (PERCELL) { const uint2 cs = __ldg(&sc.scale[cell2]); Cm2 = cs.x; sh2 = cs.y; }
                } else {
                    const u64 xi = draw_index(Xe);
                    const u32 x0 = cell & 0xFFFFu, y0 = cell >> 16;
                    for (u32 r0 = (flags & 4u) ? 1u : 0u; r0 < NS_MAX_RESAMPLE; r0 += NS_TAIL_ATTEMPTS) {
                        u32 c2 = 0, d = 0, pf = 0;
                        uint2 cs = make_uint2(Cm, sh);
                        if (lane < NS_TAIL_ATTEMPTS) {
                            const u64 x = draw_disp(Xe, r0 + lane);
                            const u32 xx = wrap_add(x0, gauss_disp(gl, (u32)(x >> 32)), sc.width);
                            const u32 yy = wrap_add(y0, gauss_disp(gl, (u32)x), sc.height);
                            const u32 ci = yy * sc.width + xx;
                            c2 = (yy << 16) | xx;
                            d = cell_deme(sc, ci);
                            pf = cell_prefix(sc, ci);                       // speculative: same round trip as the habitat test
                            if (PERCELL) cs = __ldg(&sc.scale[ci]);
                        }
                        const u32 okm = __ballot_sync(NS_FULL, lane < NS_TAIL_ATTEMPTS && d > 0);
                        if (okm) {
                            const int w = __ffs(okm) - 1;    // first accepted attempt = the sequential algorithm's choice
                            c2 = __shfl_sync(NS_FULL, c2, w); d = __shfl_sync(NS_FULL, d, w); pf = __shfl_sync(NS_FULL, pf, w);
                            Cm2 = __shfl_sync(NS_FULL, cs.x, w); sh2 = __shfl_sync(NS_FULL, cs.y, w);
                            cell2 = c2;
                            loc2 = pf + ((d == 1u) ? 0u : mulhi64_u32(xi, d));
                            c_resamples += r0 + (u32)w;
                            ok = true;
                            break;
                        }
                    }
                }
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
    if (lane == 0) {
        if (c_events) atomicAdd((unsigned long long *)&bf.ctr->n_events, c_events);
        if (c_culled) atomicAdd((unsigned long long *)&bf.ctr->n_culled, c_culled);
        if (c_resamples) atomicAdd((unsigned long long *)&bf.ctr->resamples, c_resamples);
    }
}

}  // namespace necsim
