// tail_kernel.cuh -- low-latency simulate kernel for the sequential tail: ONE lineage per warp.
//
// At low nu the last lineages are serial chains of ~1/nu events each ("its curve
// never flattens"); with a few thousand lineages left the machine is bound by the latency of one event, not by
// throughput. Every draw is a pure function of its key (seed, loc, k, j, lane) -- PAPER.md 5.2.1, L693-707 --
// so the 32 lanes of a warp may evaluate candidate draws of ONE lineage speculatively and in parallel; the
// result is identical by construction (tests/test_gpu_invariance.py runs both kernels on the same inputs):
//   - event-time search: lanes 0..15 draw the points j = 1..16 of interval k (segmented prefix sum gives the
//     partial sums T_j), lanes 16..31 draw the FIRST point of intervals k+1..k+16 (the event if interval k is
//     exhausted: a fresh interval's first point is its next event, L719-729);
//   - event: the duplicate-culling exchange is issued by lane 0 first; the speciation draw, the index draw and
//     eight dispersal attempts r..r+7 (with their habitat / prefix / turnover-scale gathers) proceed meanwhile.
#pragma once
#include "sim_kernel.cuh"

namespace necsim {

#define NS_TAIL_ATTEMPTS 8u

template <int KIND, bool DEDUP>
__global__ void __launch_bounds__(256) tail_kernel(const ScenarioDev sc, const SimBuffers bf, const EpochArgs ep) {
    __shared__ unsigned short sQ[512];
    __shared__ u64 sA[512];
    __shared__ u32 sG[KIND == 3 ? 1024 : 1];
    __shared__ unsigned short sGuide[KIND == 3 ? 256 : 1];
    for (u32 i = threadIdx.x; i < 512; i += blockDim.x) { sQ[i] = NEGLOG_Q_DEV[i]; sA[i] = NEGLOG_A_DEV[i]; }
    if (KIND == 3) gauss_stage(sc, sG, sGuide);
    __syncthreads();
    GaussLut gl; gl.tg = sG; gl.guide = sGuide; gl.R = sc.R;

    const u32 lane = threadIdx.x & 31u, half = lane >> 4, sub = lane & 15u;
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
        if (sc.per_cell_turnover) { uint2 cs = __ldg(&sc.scale[cell]); Cm = cs.x; sh = cs.y; }

        for (;;) {   // one iteration = one search round (+ the event it finds)
            if (k == ep.k_stop) {   // epoch horizon: survivor
                if (lane == 0) bf.q_out[atomicAdd(&bf.ctr->q_out, 1u)] = make_uint4(id, loc, cell, steps);
                break;
            }
            // ---- S1: speculative event-time search ---------------------------------------------------------
            const u64 kk64 = (u64)k + (half ? (u64)(1u + sub) : 0ull);
            const bool kvalid = kk64 < (u64)ep.k_stop;                     // never look at or past the horizon
            u64 X = prime(ep.key, loc, (u32)kk64) + (u64)(half ? 1u : sub + 1u) * NS_GAMMA;
            u64 T = scale_exp(neglog(draw_time(X), sQ, sA), Cm, sh);
            if (!half) {   // partial sums T_j over the 16 lanes of half 0 (half 1 keeps single draws)
#pragma unroll
                for (int o = 1; o < 16; o <<= 1) {
                    u64 t = __shfl_up_sync(0x0000FFFFu, T, o, 16);
                    if ((int)sub >= o) T += t;
                }
            }
            const bool inside = T < NS_TWO48;
            const u32 evm = __ballot_sync(NS_FULL, inside && (half ? kvalid : ((i64)T > f_last)));
            const u32 crm = __ballot_sync(NS_FULL, !inside);
            u32 j;
            u64 Te, Xe;
            if (evm & 0xFFFFu) {                       // next event is in interval k
                const int src = __ffs(evm & 0xFFFFu) - 1;
                j = (u32)src + 1u;
                Te = __shfl_sync(NS_FULL, T, src); Xe = __shfl_sync(NS_FULL, X, src);
            } else if (crm & 0xFFFFu) {                // interval k exhausted (L719, L727): first non-empty interval after it
                const u32 gap = ep.k_stop - 1u - k;                     // k < k_stop here
                const u32 nvalid = gap < 16u ? gap : 16u;   // speculated intervals before the horizon
                const u32 hm = evm >> 16;
                if (hm) {
                    const int s1 = __ffs(hm) - 1;
                    k = k + 1u + (u32)s1; j = 1u;
                    Te = __shfl_sync(NS_FULL, T, 16 + s1); Xe = __shfl_sync(NS_FULL, X, 16 + s1);
                } else {                               // all speculated intervals empty (or beyond the horizon)
                    k = k + 1u + nvalid; f_last = -1;
                    continue;
                }
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
                j = jc; Te = Tc; Xe = Xc;
            }

            // ---- event (loc, k, j) at offset Te ----------------------------------------------------------------
            uint4 old = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
            if (DEDUP && lane == 0) old = atomic_exch_128(&bf.cache[cache_slot(loc, k, j, bf.cache_mask)], make_uint4(loc, k, j, id));
            const bool can_speciate = !(KIND == 1 && cell == 0);
            const bool speciates = can_speciate && bern(draw_spec(Xe), ep.thr_nu);   // every lane, uniform
            u32 loc2 = loc, cell2 = cell, Cm2 = Cm, sh2 = sh;
            bool ok = true;
            if (!speciates) {
                if (KIND != 3) {
                    u32 rs = 0;
                    ok = disperse<KIND>(sc, ep.thr_m, Xe, cell, loc2, cell2, gl, rs);   // uniform: every lane computes the same
                    if (sc.per_cell_turnover) { uint2 cs = __ldg(&sc.scale[cell2]); Cm2 = cs.x; sh2 = cs.y; }
                } else {
                    u32 x0, y0;
                    if (sc.width_shift != 0xFFFFFFFFu) { x0 = cell & (sc.width - 1); y0 = cell >> sc.width_shift; }
                    else { y0 = cell / sc.width; x0 = cell - y0 * sc.width; }
                    const u64 xi = draw_index(Xe);
                    ok = false;
                    for (u32 r0 = 0; r0 < NS_MAX_RESAMPLE; r0 += NS_TAIL_ATTEMPTS) {
                        u32 c2 = 0, d = 0, pf = 0;
                        uint2 cs = make_uint2(Cm, sh);
                        if (lane < NS_TAIL_ATTEMPTS) {   // attempt r0 + lane (R16: redraw the whole (dx, dy) pair)
                            const u64 x = draw_disp(Xe, r0 + lane);
                            const int dx = gauss_disp(gl, (u32)(x >> 32)), dy = gauss_disp(gl, (u32)x);
                            int xx = (int)x0 + dx, yy = (int)y0 + dy;
                            if (xx < 0) xx += (int)sc.width; else if (xx >= (int)sc.width) xx -= (int)sc.width;
                            if (yy < 0) yy += (int)sc.height; else if (yy >= (int)sc.height) yy -= (int)sc.height;
                            c2 = (u32)yy * sc.width + (u32)xx;
                            d = cell_deme(sc, c2);
                            pf = cell_prefix(sc, c2);                       // speculative: same round trip as the habitat test
                            if (sc.per_cell_turnover) cs = __ldg(&sc.scale[c2]);
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
            if (DEDUP) {
                old.x = __shfl_sync(NS_FULL, old.x, 0); old.y = __shfl_sync(NS_FULL, old.y, 0);
                old.z = __shfl_sync(NS_FULL, old.z, 0); old.w = __shfl_sync(NS_FULL, old.w, 0);
                if (old.x == loc && old.y == k && old.z == j && old.w != id) {   // duplicate of a lineage that was here first
                    if (lane == 0) {
                        bf.parent[id] = old.w; bf.state[id] = 2;
                        bf.term_loc[id] = loc; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = Te; bf.steps[id] = steps;
                    }
                    c_culled++;
                    break;
                }
            }
            f_last = (i64)Te; steps++; c_events++;
            if (speciates) {
                if (lane == 0) {
                    bf.state[id] = 1;
                    bf.term_loc[id] = loc; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = Te; bf.steps[id] = steps;
                    bf.spec_ring[atomicAdd(&bf.ctr->n_spec, 1u)] = id;
                    atomicMax(&bf.ctr->j_max, j);
                }
                break;
            }
            if (!ok) { if (lane == 0) atomicMax(&bf.ctr->error, 3u); break; }
            loc = loc2; cell = cell2; Cm = Cm2; sh = sh2;
            if (ep.max_steps && steps >= ep.max_steps) {
                if (lane == 0) {
                    bf.state[id] = 3;
                    bf.term_loc[id] = loc; bf.term_k[id] = k; bf.term_j[id] = j; bf.term_f[id] = Te; bf.steps[id] = steps;
                }
                break;
            }
        }
    }
    if (lane == 0) {
        if (c_events) atomicAdd((unsigned long long *)&bf.ctr->n_events, c_events);
        if (c_culled) atomicAdd((unsigned long long *)&bf.ctr->n_culled, c_culled);
        if (c_resamples) atomicAdd((unsigned long long *)&bf.ctr->resamples, c_resamples);
    }
}

}  // namespace necsim
