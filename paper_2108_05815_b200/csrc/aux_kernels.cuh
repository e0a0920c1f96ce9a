// aux_kernels.cuh -- S0 (sample mask -> lineage queue) and S6 (resolve, radix sort, unique, labels).
// PAPER.md L2162 (population generation), L958-967 (a-posteriori coalescence: duplicates of an event are
// adjacent after sorting), L276 / L890-900 (species = distinct speciation events).
#pragma once
#include "../../include/necsim.h"
#include "sim_kernel.cuh"

namespace necsim {

#define NS_CHUNK 4096u   // mask bytes per block in the compaction kernels (256 threads x 16 bytes)

// the `cell` word of a queue entry: the cell index, or packed (y << 16 | x) for EXPLICIT_GAUSSIAN
__device__ __forceinline__ u32 queue_cell(const ScenarioDev &sc, u32 loc) {
    const u32 c = cell_of_loc(sc, loc);
    return sc.kind == 3 ? pack_xy(sc, c) : c;
}

// temporally varying habitat: the i-th present-day individual sits at (cell, i') of the present map; its indexed
// location is canonical on the oldest map: prefix[cell] + i'
__device__ __forceinline__ u32 era_start_loc(const ScenarioDev &sc, u32 i) {
    u32 lo = 0, hi = sc.ncells;                      // invariant: prefix0[lo] <= i < prefix0[hi]
    while (hi - lo > 1) { u32 mid = lo + ((hi - lo) >> 1); if (sc.prefix0[mid] <= i) lo = mid; else hi = mid; }
    return sc.prefix[lo] + (i - sc.prefix0[lo]);
}

// S0, pass 1: number of sampled individuals per chunk
__global__ void __launch_bounds__(256) mask_count_kernel(const uint8_t *__restrict__ mask, u64 n, u32 *__restrict__ chunk_count) {
    __shared__ u32 wsum[8];
    u64 base = (u64)blockIdx.x * NS_CHUNK + (u64)threadIdx.x * 16u;
    u32 c = 0;
    for (u32 t = 0; t < 16; ++t) { u64 i = base + t; if (i < n && mask[i]) ++c; }
    for (int o = 16; o; o >>= 1) c += __shfl_down_sync(NS_FULL, c, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) { u32 s = 0; for (int w = 0; w < 8; ++w) s += wsum[w]; chunk_count[blockIdx.x] = s; }
}

// exclusive scan of a u32 array by one block (n up to a few 10^5); total -> *total_out (may be NULL)
__global__ void __launch_bounds__(1024) scan_exclusive_kernel(u32 *__restrict__ a, u32 n, u32 *__restrict__ total_out) {
    __shared__ u32 wsum[32];
    __shared__ u32 carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const u32 lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    for (u32 start = 0; start < n; start += 1024u) {
        u32 i = start + threadIdx.x;
        u32 v = i < n ? a[i] : 0u, x = v;
        for (int o = 1; o < 32; o <<= 1) { u32 y = __shfl_up_sync(NS_FULL, x, o); if ((int)lane >= o) x += y; }
        if (lane == 31) wsum[w] = x;
        __syncthreads();
        if (w == 0) {
            u32 s = wsum[lane], t = s;
            for (int o = 1; o < 32; o <<= 1) { u32 y = __shfl_up_sync(NS_FULL, t, o); if ((int)lane >= o) t += y; }
            wsum[lane] = t - s;   // exclusive warp offsets
        }
        __syncthreads();
        u32 excl = carry + wsum[w] + (x - v);
        if (i < n) a[i] = excl;
        __syncthreads();
        if (threadIdx.x == 1023) carry = excl + v;
        __syncthreads();
    }
    if (threadIdx.x == 0 && total_out) *total_out = carry;
}

// exclusive scan of a long u32 array in three launches: per-block scans of 8192 elements + their totals, a scan of the totals
// (scan_exclusive_kernel), and the add-back
#define NS_SCAN_TILE 8192u
__global__ void __launch_bounds__(1024) scan_tile_kernel(u32 *__restrict__ a, u32 n, u32 *__restrict__ sums) {
    __shared__ u32 wsum[32];
    const u32 lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const u32 base = blockIdx.x * NS_SCAN_TILE + threadIdx.x * 8u;
    u32 v[8], t = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { v[q] = (base + q < n) ? a[base + q] : 0u; t += v[q]; }
    u32 x = t;
    for (int o = 1; o < 32; o <<= 1) { u32 y = __shfl_up_sync(NS_FULL, x, o); if ((int)lane >= o) x += y; }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
        u32 s = wsum[lane], z = s;
        for (int o = 1; o < 32; o <<= 1) { u32 y = __shfl_up_sync(NS_FULL, z, o); if ((int)lane >= o) z += y; }
        wsum[lane] = z - s;
        if (lane == 31) sums[blockIdx.x] = z;
    }
    __syncthreads();
    u32 run = wsum[w] + (x - t);
#pragma unroll
    for (int q = 0; q < 8; ++q) { if (base + q < n) a[base + q] = run; run += v[q]; }
}
__global__ void __launch_bounds__(1024) scan_add_kernel(u32 *__restrict__ a, u32 n, const u32 *__restrict__ sums) {
    const u32 base = blockIdx.x * NS_SCAN_TILE + threadIdx.x * 8u, add = sums[blockIdx.x];
#pragma unroll
    for (int q = 0; q < 8; ++q) if (base + q < n) a[base + q] += add;
}

// S0, pass 2: ordered compaction -> queue entries {id, loc, cell, steps = 0}; id = rank in ascending loc
__global__ void __launch_bounds__(256) mask_scatter_kernel(const ScenarioDev sc, const uint8_t *__restrict__ mask, u64 n,
                                                           const u32 *__restrict__ chunk_offset, uint4 *__restrict__ queue, u32 capacity) {
    __shared__ u32 wsum[8];
    u64 base = (u64)blockIdx.x * NS_CHUNK + (u64)threadIdx.x * 16u;
    u32 bits = 0;
    for (u32 t = 0; t < 16; ++t) { u64 i = base + t; if (i < n && mask[i]) bits |= 1u << t; }
    u32 c = __popc(bits), x = c;
    const u32 lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { u32 y = __shfl_up_sync(NS_FULL, x, o); if ((int)lane >= o) x += y; }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    u32 off = chunk_offset[blockIdx.x] + (x - c);
    for (u32 ww = 0; ww < w; ++ww) off += wsum[ww];
    while (bits) {
        u32 t = __ffs(bits) - 1; bits &= bits - 1;
        u32 loc = (u32)(base + t);
        if (sc.n_eras) loc = era_start_loc(sc, loc);
        if (off < capacity) queue[off] = make_uint4(off, loc, queue_cell(sc, loc), 0u);
        ++off;
    }
}

// S0 without a mask: everyone is sampled
__global__ void __launch_bounds__(256) all_sampled_kernel(const ScenarioDev sc, u32 n, uint4 *__restrict__ queue) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { const u32 loc = sc.n_eras ? era_start_loc(sc, i) : i; queue[i] = make_uint4(i, loc, queue_cell(sc, loc), 0u); }
}

// ---- S6 ------------------------------------------------------------------------------------------
// 144-bit sort key (k, f, loc, j) as 18 little-endian bytes: j[0..3], loc[4..7], f[8..13], k[14..17]
__device__ __forceinline__ u32 key_byte(const SimBuffers &bf, u32 id, u32 b) {
    if (b < 4) return (bf.term_j[id] >> (8 * b)) & 255u;
    if (b < 8) return (bf.term_loc[id] >> (8 * (b - 4))) & 255u;
    if (b < 14) return (u32)(bf.term_f[id] >> (8 * (b - 8))) & 255u;
    return ((bf.term_k[id] - bf.k_base) >> (8 * (b - 14))) & 255u;
}

#define NS_SORT_TILE 2048u
// one LSD pass, step 1: per-block digit histogram, bin-major: hist[d * nblocks + block]. The digit of position i is kept in
// digit[i], so that the scatter of the same pass reads it in order instead of gathering the key through perm a second time.
__global__ void __launch_bounds__(256) radix_hist_kernel(const SimBuffers bf, const u32 *__restrict__ perm, u32 n, u32 byte,
                                                         u32 *__restrict__ hist, u32 nblocks, uint8_t *__restrict__ digit) {
    __shared__ u32 h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    u32 start = blockIdx.x * NS_SORT_TILE;
    for (u32 r = 0; r < NS_SORT_TILE; r += 256u) {
        u32 i = start + r + threadIdx.x;
        if (i < n) {
            u32 d = key_byte(bf, perm[i], byte);
            digit[i] = (uint8_t)d;
            atomicAdd(&h[d], 1u);
        }
    }
    __syncthreads();
    hist[threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}
// step 3 (after an exclusive scan of hist): stable scatter. A warp ranks 256 consecutive positions, 32 at a time, against its own
// digit counters (no block barrier inside the loop); the counters of the eight warps are then turned into write positions at once.
__global__ void __launch_bounds__(256) radix_scatter_kernel(const u32 *__restrict__ perm_in, u32 *__restrict__ perm_out, u32 n,
                                                            const u32 *__restrict__ hist, u32 nblocks, const uint8_t *__restrict__ digit) {
    __shared__ u32 wcount[8][256];
    const u32 lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    for (u32 ww = 0; ww < 8; ++ww) wcount[ww][threadIdx.x] = 0;
    __syncthreads();
    const u32 start = blockIdx.x * NS_SORT_TILE + w * (NS_SORT_TILE / 8u);
    u32 item[8], dr[8];                                 // dr = digit | rank inside the warp's 256 positions << 9
#pragma unroll
    for (u32 r = 0; r < 8; ++r) {
        u32 i = start + r * 32u + lane;
        bool valid = i < n;
        item[r] = valid ? perm_in[i] : 0u;
        u32 d = valid ? (u32)digit[i] : 256u + lane;    // invalid lanes never match anyone
        u32 peers = __match_any_sync(NS_FULL, d);
        u32 before = __popc(peers & lanemask_lt());
        u32 rank = valid ? wcount[w][d] + before : 0u;
        __syncwarp();
        if (valid && before == 0) wcount[w][d] = rank + __popc(peers);
        __syncwarp();
        dr[r] = d | (rank << 9);
    }
    __syncthreads();
    u32 run = hist[threadIdx.x * nblocks + blockIdx.x];   // digit threadIdx.x: the block's base, then the warps in order
    for (u32 ww = 0; ww < 8; ++ww) { u32 c = wcount[ww][threadIdx.x]; wcount[ww][threadIdx.x] = run; run += c; }
    __syncthreads();
#pragma unroll
    for (u32 r = 0; r < 8; ++r) {
        u32 d = dr[r] & 511u;
        if (d < 256u) perm_out[wcount[w][d] + (dr[r] >> 9)] = item[r];
    }
}

__device__ __forceinline__ bool same_event(const SimBuffers &bf, u32 a, u32 b) {
    return bf.term_k[a] == bf.term_k[b] && bf.term_f[a] == bf.term_f[b] && bf.term_loc[a] == bf.term_loc[b] &&
           bf.term_j[a] == bf.term_j[b];
}
// unique, step 1: head flags over the sorted records
__global__ void __launch_bounds__(256) unique_flag_kernel(const SimBuffers bf, const u32 *__restrict__ perm, u32 n, u32 *__restrict__ flag) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) flag[i] = (i == 0 || !same_event(bf, perm[i], perm[i - 1])) ? 1u : 0u;
}
// unique, step 2 (flag scanned exclusively -> uidx): write the species table; species_of[lineage] = rank
__global__ void __launch_bounds__(256) unique_write_kernel(const SimBuffers bf, const u32 *__restrict__ perm, u32 n, const u32 *__restrict__ uidx,
                                                           necsim_event *__restrict__ events, u32 *__restrict__ species_of, double delta_t) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u32 id = perm[i];
    bool head = (i == 0) || !same_event(bf, id, perm[i - 1]);
    u32 e = head ? uidx[i] : uidx[i] - 1u;     // exclusive scan of head flags: a non-head belongs to the previous head
    species_of[id] = e;
    if (head) {
        necsim_event ev;
        ev.loc = bf.term_loc[id]; ev.k = bf.term_k[id]; ev.j = bf.term_j[id]; ev.abundance = 0;
        ev.f = bf.term_f[id]; ev.time = event_time(ev.k, ev.f, delta_t);
        events[e] = ev;
    }
}
// pointer jumping over the "culled at an event another lineage executed" links: parent <- grandparent where the parent was culled
// too. Every value a racing thread can read here is an ancestor, so the links stay a forest; k rounds divide the depth by 2^k.
__global__ void __launch_bounds__(256) parent_jump_kernel(const SimBuffers bf, u32 n) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || bf.state[i] != 2) return;
    const u32 p = bf.parent[i];
    if (bf.state[p] == 2) bf.parent[i] = bf.parent[p];
}
// resolve + label: follow the "culled at an event another lineage executed" links to a lineage that
// ended by itself (links point to earlier arrivals at one event and time increases along a lineage: a forest)
__global__ void __launch_bounds__(256) label_kernel(const SimBuffers bf, u32 n, const u32 *__restrict__ species_of, necsim_event *__restrict__ events,
                                                    u32 *__restrict__ labels) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u32 r = i;
    while (bf.state[r] == 2) r = bf.parent[r];
    if (bf.state[r] == 1) {
        u32 e = species_of[r];
        labels[i] = e;
        atomicAdd(&events[e].abundance, 1u);
    } else {
        labels[i] = 0xFFFFFFFFu;
        atomicAdd(&bf.ctr->n_unfinished, 1u);
    }
}

// ---- merge of species tables from isolated partitions -------
// AoS species records -> the SoA key arrays the radix passes read; perm = identity
__global__ void __launch_bounds__(256) merge_unpack_kernel(const necsim_event *__restrict__ in, u32 n, const SimBuffers bf, u32 *__restrict__ perm) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const necsim_event e = in[i];
    bf.term_loc[i] = e.loc; bf.term_k[i] = e.k; bf.term_j[i] = e.j; bf.term_f[i] = e.f;
    perm[i] = i;
}
// sorted + head-flag-scanned records -> merged table (abundances add up), map[input record] = rank in the merged table
__global__ void __launch_bounds__(256) merge_write_kernel(const SimBuffers bf, const u32 *__restrict__ perm, u32 n, const u32 *__restrict__ uidx,
                                                          const necsim_event *__restrict__ in, necsim_event *__restrict__ out, u32 *__restrict__ map) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const u32 id = perm[i];
    const bool head = (i == 0) || !same_event(bf, id, perm[i - 1]);
    const u32 e = head ? uidx[i] : uidx[i] - 1u;
    map[id] = e;
    if (head) { out[e].loc = in[id].loc; out[e].k = in[id].k; out[e].j = in[id].j; out[e].f = in[id].f; out[e].time = in[id].time; }
    atomicAdd(&out[e].abundance, in[id].abundance);
}

// ---- full event stream: one epoch's ring, sorted and made unique, appended to the run's stream -------
__global__ void __launch_bounds__(256) iota_kernel(u32 *perm, u32 n) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) perm[i] = i;
}
// The ring is radix-sorted on a prefix of its key only: k and the top `fbytes` bytes of f. Records that share the prefix are
// adjacent and few (redundant executions of one event, and distinct events whose offsets agree in the leading bits), so the
// first thread of such a run puts it into full (f, loc, j) order by insertion. Runs of sentinels stay as they are.
__device__ __forceinline__ bool stream_less(const SimBuffers &bf, u32 a, u32 b) {   // same k: order by (f, loc, j)
    const u64 fa = bf.term_f[a], fb = bf.term_f[b];
    if (fa != fb) return fa < fb;
    const u32 la = bf.term_loc[a], lb = bf.term_loc[b];
    if (la != lb) return la < lb;
    return bf.term_j[a] < bf.term_j[b];
}
// Also writes the head flags of the sorted ring: 1 for the first record of every distinct event, 0 for its redundant copies
// (adjacent after the sort) and for sentinel records (k = the epoch's k_stop: reserved but unused slots, sorted last).
__global__ void __launch_bounds__(256) stream_ties_kernel(const SimBuffers bf, u32 *__restrict__ perm, u32 n, u32 k_sentinel, u32 fbytes,
                                                          u32 *__restrict__ flag) {
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31u;
    const bool in = i < n;
    const u32 sh = 48u - 8u * fbytes;
    const u32 id = in ? perm[i] : 0u, k = in ? bf.term_k[id] : k_sentinel;
    const u64 fp = in ? bf.term_f[id] >> sh : 0ull;
    // the previous record's prefix comes from the neighbouring lane (a record a run's first thread is moving at this moment
    // is still one of that run: the answer is the same)
    u32 pk = __shfl_up_sync(NS_FULL, k, 1);
    u64 pf = __shfl_up_sync(NS_FULL, fp, 1);
    if (in && lane == 0 && i != 0) { const u32 pv = perm[i - 1]; pk = bf.term_k[pv]; pf = bf.term_f[pv] >> sh; }
    if (!in) return;
    if (k == k_sentinel) { flag[i] = 0u; return; }
    if (i != 0 && pk == k && pf == fp) return;   // not the first of its run
    flag[i] = 1u;
    u32 e = i + 1;
    for (; e < n; ++e) {
        const u32 x = perm[e];
        if (bf.term_k[x] != k || (bf.term_f[x] >> sh) != fp) break;
        u32 q = e;
        while (q > i && stream_less(bf, x, perm[q - 1])) { perm[q] = perm[q - 1]; --q; }
        perm[q] = x;
    }
    for (u32 p = i + 1; p < e; ++p) flag[p] = same_event(bf, perm[p], perm[p - 1]) ? 0u : 1u;
}
// bf.term_* alias the ring's key arrays; uidx = the head flags scanned exclusively, *total = their sum: the heads are written
__global__ void __launch_bounds__(256) stream_write_kernel(const SimBuffers bf, const u32 *__restrict__ rec_loc2, const u32 *__restrict__ perm, u32 n,
                                                           const u32 *__restrict__ uidx, const u32 *__restrict__ total, u64 base, u64 cap, u32 *__restrict__ s_loc,
                                                           u32 *__restrict__ s_k, u32 *__restrict__ s_j, u64 *__restrict__ s_f, u32 *__restrict__ s_loc2) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const u32 u = uidx[i], nx = (i + 1 < n) ? uidx[i + 1] : *total;
    if (nx == u) return;
    const u64 o = base + u;
    if (o >= cap) return;
    const u32 id = perm[i];
    s_loc[o] = bf.term_loc[id]; s_k[o] = bf.term_k[id]; s_j[o] = bf.term_j[id]; s_f[o] = bf.term_f[id]; s_loc2[o] = rec_loc2[id];
}

__global__ void copy_u32_kernel(u32 *a, const u32 *src, u32 n) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = src[i];
}

}  // namespace necsim
