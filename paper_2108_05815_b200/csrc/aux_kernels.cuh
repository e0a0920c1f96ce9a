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
    const bool full = base + 8u <= n;                  // (a is 32-byte aligned at base: two 16-byte loads instead of eight strided words)
    if (full) {
        const uint4 p0 = *(const uint4 *)(a + base), p1 = *(const uint4 *)(a + base + 4u);
        v[0] = p0.x; v[1] = p0.y; v[2] = p0.z; v[3] = p0.w; v[4] = p1.x; v[5] = p1.y; v[6] = p1.z; v[7] = p1.w;
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = (base + q < n) ? a[base + q] : 0u;
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) t += v[q];
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
    if (full) {
        u32 e[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) { e[q] = run; run += v[q]; }
        *(uint4 *)(a + base) = make_uint4(e[0], e[1], e[2], e[3]); *(uint4 *)(a + base + 4u) = make_uint4(e[4], e[5], e[6], e[7]);
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) { if (base + q < n) a[base + q] = run; run += v[q]; }
    }
}
__global__ void __launch_bounds__(1024) scan_add_kernel(u32 *__restrict__ a, u32 n, const u32 *__restrict__ sums) {
    const u32 base = blockIdx.x * NS_SCAN_TILE + threadIdx.x * 8u, add = sums[blockIdx.x];
    if (base + 8u <= n) {
        uint4 p0 = *(const uint4 *)(a + base), p1 = *(const uint4 *)(a + base + 4u);
        p0.x += add; p0.y += add; p0.z += add; p0.w += add; p1.x += add; p1.y += add; p1.z += add; p1.w += add;
        *(uint4 *)(a + base) = p0; *(uint4 *)(a + base + 4u) = p1;
        return;
    }
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
// The ring holds one 32-byte record per executed event and, beside it, the record's 64-bit time key (k - k_start) << 40 | f >> 8.
// The sort never touches the records: LSD radix passes over (key, index) pairs, 12 bytes read and 12 written per record and pass,
// fully coalesced; only k and the leading `fbytes` bytes of f are sorted on. Records that agree there are adjacent and few (redundant
// executions of one event, and distinct events whose offsets share those bits); the first thread of such a run orders it by the full
// (f, loc, j) with the records gathered through the index (one 32-byte sector each). Runs longer than NS_RUN_INLINE go to a warp.
#define NS_RUN_INLINE 16u
#define NS_PAIR_TILE 4096u          // pairs per block and pass: 16 per digit on average, so that a digit's pairs leave the block as one run
// Keys: the ring's 64-bit keys, or (compact sort) 32-bit keys ck = (u32)(key >> cshift) that hold the interval and the leading bits of
// f in one word: 8-byte pairs instead of 12-byte ones. The first compact pass reads the 64-bit keys and writes the 32-bit ones.
template <typename KIN>
__global__ void __launch_bounds__(256) pair_hist_kernel(const KIN *__restrict__ keys, u32 n, u32 cshift, u32 shift, u32 *__restrict__ hist, u32 nblocks) {
    __shared__ u32 h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const u32 start = blockIdx.x * NS_PAIR_TILE;
    u32 d[NS_PAIR_TILE / 256u];
#pragma unroll
    for (u32 r = 0; r < NS_PAIR_TILE / 256u; ++r) {   // all loads of the thread in flight before the first atomic
        const u32 i = start + r * 256u + threadIdx.x;
        d[r] = i < n ? (u32)((keys[i] >> cshift) >> shift) & 255u : 256u;
    }
#pragma unroll
    for (u32 r = 0; r < NS_PAIR_TILE / 256u; ++r) if (d[r] < 256u) atomicAdd(&h[d[r]], 1u);
    __syncthreads();
    hist[threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}
// stable scatter of the pairs (after an exclusive scan of hist); idx_in == NULL: the identity (first pass). A warp ranks its 256
// consecutive pairs against its own digit counters, the block orders the tile by digit in shared memory, and every digit's pairs
// are then written to their place in one coalesced run (a direct scatter from registers writes 8 useful bytes per 32-byte sector).
// 512 threads x 8 pairs: with 16 pairs per thread in registers the kernel ran two blocks of 256 threads per SM (25 % of the warp slots,
// 14 % of the issue slots, 25 % of the HBM peak: ncu, profiles/r2_ncu_stream_kernels_c6.md); now three blocks of 512.
#define NS_PAIR_THREADS 512u
#define NS_PAIR_WARPS (NS_PAIR_THREADS / 32u)
#define NS_PAIR_ROUNDS (NS_PAIR_TILE / NS_PAIR_THREADS)
template <typename KIN, typename KOUT>
__global__ void __launch_bounds__(NS_PAIR_THREADS, 3) pair_scatter_kernel(const KIN *__restrict__ keys_in, const u32 *__restrict__ idx_in, KOUT *__restrict__ keys_out,
                                                                          u32 *__restrict__ idx_out, u32 n, u32 cshift, u32 shift, const u32 *__restrict__ hist, u32 nblocks) {
    extern __shared__ __align__(16) unsigned char pair_smem[];
    KOUT *skey = (KOUT *)pair_smem;                         // [NS_PAIR_TILE]
    u32 *sidx = (u32 *)(skey + NS_PAIR_TILE);               // [NS_PAIR_TILE]
    u32 (*wcount)[256] = (u32 (*)[256])(sidx + NS_PAIR_TILE);   // [NS_PAIR_WARPS][256]
    u32 *bdo = (u32 *)(wcount + NS_PAIR_WARPS);             // [256] first position of a digit inside the ordered tile
    u32 *gbase = bdo + 256;                                 // [256] global position of the tile's first pair of a digit
    u32 *wtot = gbase + 256;                                // [8]
    const u32 lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    for (u32 t = threadIdx.x; t < NS_PAIR_WARPS * 256u; t += NS_PAIR_THREADS) (&wcount[0][0])[t] = 0;
    __syncthreads();
    const u32 tile0 = blockIdx.x * NS_PAIR_TILE, start = tile0 + w * (NS_PAIR_TILE / NS_PAIR_WARPS);
    KOUT key[NS_PAIR_ROUNDS];
    u32 item[NS_PAIR_ROUNDS], dr[NS_PAIR_ROUNDS];       // dr = digit | rank inside the warp's 256 positions << 9
#pragma unroll
    for (u32 r = 0; r < NS_PAIR_ROUNDS; ++r) {          // the loads first: all of a thread's pairs are in flight together
        const u32 i = start + r * 32u + lane;
        const bool valid = i < n;
        key[r] = valid ? (KOUT)(keys_in[i] >> cshift) : (KOUT)0;
        item[r] = valid ? (idx_in ? idx_in[i] : i) : 0u;
    }
#pragma unroll
    for (u32 r = 0; r < NS_PAIR_ROUNDS; ++r) {
        const bool valid = start + r * 32u + lane < n;
        const u32 d = valid ? (u32)(key[r] >> shift) & 255u : 256u + lane;    // invalid lanes never match anyone
        const u32 peers = __match_any_sync(NS_FULL, d);
        const u32 before = __popc(peers & lanemask_lt());
        const u32 rank = valid ? wcount[w][d] + before : 0u;
        __syncwarp();
        if (valid && before == 0) wcount[w][d] = rank + __popc(peers);
        __syncwarp();
        dr[r] = d | (rank << 9);
    }
    __syncthreads();
    // digit threadIdx.x (threads 0..255): the tile's count, the warps' offsets inside the digit, the digit's first position in the ordered tile
    u32 tot = 0, x = 0;
    if (threadIdx.x < 256u) {
        for (u32 ww = 0; ww < NS_PAIR_WARPS; ++ww) { const u32 c = wcount[ww][threadIdx.x]; wcount[ww][threadIdx.x] = tot; tot += c; }
        x = tot;                                        // exclusive scan of the 256 digit counts over the first 8 warps
        for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(NS_FULL, x, o); if ((int)lane >= o) x += y; }
        if (lane == 31) wtot[w] = x;
    }
    __syncthreads();
    if (threadIdx.x < 256u) {
        u32 off = x - tot;
        for (u32 ww = 0; ww < w; ++ww) off += wtot[ww];
        bdo[threadIdx.x] = off;
        gbase[threadIdx.x] = hist[threadIdx.x * nblocks + blockIdx.x];
    }
    __syncthreads();
#pragma unroll
    for (u32 r = 0; r < NS_PAIR_ROUNDS; ++r) {
        const u32 d = dr[r] & 511u;
        if (d < 256u) { const u32 p = bdo[d] + wcount[w][d] + (dr[r] >> 9); skey[p] = key[r]; sidx[p] = item[r]; }
    }
    __syncthreads();
    const u32 cnt = min(NS_PAIR_TILE, n - tile0);
    for (u32 t = threadIdx.x; t < cnt; t += NS_PAIR_THREADS) {
        const KOUT k = skey[t];
        const u32 d = (u32)(k >> shift) & 255u;
        const u32 o = gbase[d] + (t - bdo[d]);
        keys_out[o] = k; idx_out[o] = sidx[t];
    }
}
#define NS_PAIR_SMEM(keybytes) (NS_PAIR_TILE * ((keybytes) + 4u) + NS_PAIR_WARPS * 256u * 4u + 2u * 256u * 4u + 64u)
// order of two records of the same interval k: by (f, loc, j)
__device__ __forceinline__ bool rec_less(const uint4 *__restrict__ rec, u32 a, u32 b) {
    const uint4 a1 = rec[2u * a + 1u], b1 = rec[2u * b + 1u];
    const u64 fa = ((u64)a1.y << 32) | a1.x, fb = ((u64)b1.y << 32) | b1.x;
    if (fa != fb) return fa < fb;
    const uint4 a0 = rec[2u * a], b0 = rec[2u * b];
    if (a0.x != b0.x) return a0.x < b0.x;
    return a0.z < b0.z;
}
__device__ __forceinline__ bool rec_same(const uint4 *__restrict__ rec, u32 a, u32 b) {
    const uint4 a0 = rec[2u * a], b0 = rec[2u * b], a1 = rec[2u * a + 1u], b1 = rec[2u * b + 1u];
    return a0.x == b0.x && a0.y == b0.y && a0.z == b0.z && a1.x == b1.x && a1.y == b1.y;
}
// Runs of equal key prefix (key >> pshift): head flags (1 = first record of a distinct event; redundant copies, adjacent after the
// sort, and sentinels get 0) and the full order inside a run. Only the first thread of a run writes idx[i..e) and
// flag[i..e); everybody else reads the keys, which this kernel never changes. Long runs are queued for stream_long_runs_kernel.
template <typename K>
__global__ void __launch_bounds__(256) stream_ties_kernel(const K *__restrict__ keys, u32 *__restrict__ idx, const uint4 *__restrict__ rec, u32 n, u32 pshift,
                                                          uint8_t *__restrict__ flag, u32 *__restrict__ long_runs, u32 *__restrict__ n_long, u32 long_cap) {
    const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const K key = keys[i];
    if (key == (K)~(K)0) { flag[i] = 0u; return; }       // reserved but unused ring slot
    const K kp = key >> pshift;
    if (i != 0 && (keys[i - 1] >> pshift) == kp) return; // not the first of its run
    u32 e = i + 1;
    while (e < n && (keys[e] >> pshift) == kp) ++e;
    if (e == i + 1) { flag[i] = 1u; return; }            // the usual case: nothing shares the prefix
    if (e - i > NS_RUN_INLINE) {
        const u32 slot = atomicAdd(n_long, 1u);
        if (slot < long_cap) { long_runs[2u * slot] = i; long_runs[2u * slot + 1u] = e - i; return; }
    }
    for (u32 p = i + 1; p < e; ++p) {                    // insertion sort of idx[i..e) by (f, loc, j)
        const u32 x = idx[p];
        u32 q = p;
        while (q > i && rec_less(rec, x, idx[q - 1])) { idx[q] = idx[q - 1]; --q; }
        idx[q] = x;
    }
    flag[i] = 1u;
    for (u32 p = i + 1; p < e; ++p) flag[p] = rec_same(rec, idx[p], idx[p - 1]) ? 0u : 1u;
}
// One warp per long run. Long runs are almost always copies of ONE event (many lineages on a shared path, dedup off or a small
// cache): that is checked first in a single sweep. Otherwise the run is ordered by ranking every record against all others.
__global__ void __launch_bounds__(256) stream_long_runs_kernel(u32 *__restrict__ idx, const uint4 *__restrict__ rec, uint8_t *__restrict__ flag,
                                                               const u32 *__restrict__ long_runs, const u32 *__restrict__ n_long, u32 long_cap, u32 *__restrict__ tmp) {
    const u32 lane = threadIdx.x & 31u, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const u32 nl = min(*n_long, long_cap);
    for (u32 r = warp; r < nl; r += nwarps) {
        const u32 i = long_runs[2u * r], L = long_runs[2u * r + 1u];
        const u32 first = idx[i];
        bool same = true;
        for (u32 p = lane; p < L; p += 32u) same = same && rec_same(rec, idx[i + p], first);
        if (__all_sync(NS_FULL, same)) {
            for (u32 p = lane; p < L; p += 32u) flag[i + p] = p == 0u ? 1u : 0u;
            continue;
        }
        for (u32 p = lane; p < L; p += 32u) {            // rank of record p: records before it in (f, loc, j), ties by position
            const u32 x = idx[i + p];
            u32 rank = 0;
            for (u32 q = 0; q < L; ++q) {
                const u32 y = idx[i + q];
                if (rec_less(rec, y, x) || (q < p && !rec_less(rec, x, y))) ++rank;
            }
            tmp[i + rank] = x;
        }
        __syncwarp();
        for (u32 p = lane; p < L; p += 32u) idx[i + p] = tmp[i + p];
        __syncwarp();
        for (u32 p = lane; p < L; p += 32u) flag[i + p] = (p == 0u || !rec_same(rec, idx[i + p], idx[i + p - 1u])) ? 1u : 0u;
    }
}
// The head flags are bytes. A block owns NS_WRITE_TILE consecutive records: stream_count_kernel sums their flags into bsum[block], the
// host scans bsum (one entry per 2048 records instead of a scan over one word per record), stream_write_kernel recomputes the positions
// inside its tile with ballots and appends the heads to the stream (SoA, coalesced writes; the 32-byte records come through the index).
#define NS_WRITE_TILE 2048u
__global__ void __launch_bounds__(256) stream_count_kernel(const uint8_t *__restrict__ flag, u32 n, u32 *__restrict__ bsum) {
    __shared__ u32 ws[8];
    const u32 i0 = blockIdx.x * NS_WRITE_TILE + threadIdx.x * 8u;
    u32 c = 0;
    if (i0 + 8u <= n) { const uint2 v = *(const uint2 *)(flag + i0); c = __popc(v.x & 0x01010101u) + __popc(v.y & 0x01010101u); }
    else for (u32 t = i0; t < n; ++t) c += flag[t] & 1u;
    for (int o = 16; o; o >>= 1) c += __shfl_down_sync(NS_FULL, c, o);
    if ((threadIdx.x & 31u) == 0) ws[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) { u32 t = 0; for (u32 w = 0; w < 8; ++w) t += ws[w]; bsum[blockIdx.x] = t; }
}
__global__ void __launch_bounds__(256) stream_write_kernel(const uint4 *__restrict__ rec, const u32 *__restrict__ idx, u32 n, const uint8_t *__restrict__ flag,
                                                           const u32 *__restrict__ bsum, u64 base, u64 cap, u32 *__restrict__ s_loc,
                                                           u32 *__restrict__ s_k, u32 *__restrict__ s_j, u64 *__restrict__ s_f, u32 *__restrict__ s_loc2) {
    __shared__ u32 ws[8];
    const u32 lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    u32 run = bsum[blockIdx.x];                          // heads before this block (bsum is scanned exclusively)
    for (u32 sub = 0; sub < NS_WRITE_TILE; sub += 256u) {
        const u32 i = blockIdx.x * NS_WRITE_TILE + sub + threadIdx.x;
        const bool head = i < n && (flag[i] & 1u);
        const u32 b = __ballot_sync(NS_FULL, head);
        if (lane == 0) ws[w] = __popc(b);
        __syncthreads();
        u32 woff = 0, tot = 0;
        for (u32 q = 0; q < 8; ++q) { const u32 c = ws[q]; if (q < w) woff += c; tot += c; }
        __syncthreads();
        if (head) {
            const u64 o = base + run + woff + __popc(b & lanemask_lt());
            if (o < cap) {
                const u32 id = idx[i];
                const uint4 r0 = rec[2u * id], r1 = rec[2u * id + 1u];
                s_loc[o] = r0.x; s_k[o] = r0.y; s_j[o] = r0.z; s_loc2[o] = r0.w; s_f[o] = ((u64)r1.y << 32) | r1.x;
            }
        }
        run += tot;
    }
}

__global__ void copy_u32_kernel(u32 *a, const u32 *src, u32 n) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = src[i];
}

}  // namespace necsim
