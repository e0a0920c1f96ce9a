// sim_types.cuh -- plain structs passed by value to the kernels (constants live in the kernel
// parameter bank, the analogue of the paper's PTX-JIT constant folding).
#pragma once
#include "device_prims.cuh"

namespace necsim {

// Device view of a scenario (tables live in the caller's scenario workspace).
struct ScenarioDev {
    int kind;
    u32 width, height, ncells;
    u32 width_shift;           // log2(width) if width is a power of two, else 0xFFFFFFFF
    u32 uniform_deme;          // != 0: every cell has this deme (host / init only; explicit kinds always carry the tables)
    u32 per_cell_turnover;     // 0: Cm_u/sh_u apply everywhere
    u32 Cm_u, sh_u;
    u64 n_locations;           // all indexed locations
    u64 n_sampleable;          // domain of the sample mask
    u32 J_local, J_meta;       // spatially implicit
    const uint8_t *hab8;       // [ncells] min(deme, 255)
    const u32 *deme32;         // [ncells] full deme (read only where hab8 == 255)
    const u32 *prefix;         // [ncells+1] exclusive prefix sum of deme
    // compact habitat table (EXPLICIT_GAUSSIAN whose habitat cells all hold `compact_deme` individuals; NULL otherwise): per
    // 32-cell block of a row {habitat bit mask, prefix sum at the block's first cell}. deme and prefix of a cell come out of
    // ONE 8-byte read: deme = bit ? compact_deme : 0, prefix = base + compact_deme * popc(mask below the bit). 128x smaller
    // than hab8 + prefix (C5: 4 MB instead of 84 MB), so a lineage's neighbourhood stays in L1 and the table in L2.
    // Tiled: entry of block b of row y at ((y / 16) * nbx + b) * 16 + y % 16, i.e. one 128-byte line holds the same block of 16
    // consecutive rows. The 32 gathers of a tail round (targets within a few sigma of one origin) then touch a handful of lines
    // instead of one line per row: a warp's gather is served line by line.
    const uint2 *hab64;        // [ceil(height / 16) * nbx * 16]
    u32 nbx;                   // 32-cell blocks per row = ceil(width / 32)
    u32 compact_deme;
    const uint2 *scale;        // [ncells] (Cm, sh) when per_cell_turnover
    const uint2 *alias;        // [ncells*ncells] (thresh, alias) for EXPLICIT_MATRIX
    const u64 *pois;           // [256] Poisson cdf thresholds of mu_max (sampler 1)
    const u32 *thin;           // [ncells] thinning thresholds (sampler 1 with per-cell turnover)
    u32 sampler;               // 0 exponential, 1 Poisson / order statistics
    const u32 *gauss;          // [gauss_len] rounded-normal thresholds, padded with 0xFFFFFFFF to a power of two
    int R;                     // displacement range: dx in [-R, R]
    u32 gauss_len;             // power of two >= 2R
    double delta_t;
    // temporally varying habitat: n_eras > 0 -> era e holds for k >= era_start[e] (era_start[0] = 0, unused entries
    // 0xFFFFFFFF). hab8 / deme32 / prefix are then those of the OLDEST map (locations are canonical on it); era_hab8[e * ncells + cell]
    // (and era_deme32 where a deme >= 255) is the map the dispersal of an event of era e is tested against; prefix0 = prefix sums of
    // the present-day map (S0: the sample mask ranges over the present-day individuals).
    u32 n_eras;
    u32 era_start[4];
    const uint8_t *era_hab8;
    const u32 *era_deme32;
    const u32 *prefix0;
    float margin;              // search filter (exponential sampler): NS_MARGIN * (1 + 1/mu_min), mu_min over the habitat cells
};

// Device counters of one simulate call (zeroed at its start). 64-bit where they can exceed 2^32.
struct SimCounters {
    u32 q_head;                // next entry of the input queue to hand out
    u32 q_out;                 // entries written to the output queue (survivors of this epoch)
    u32 n_spec;                // speciation records in the ring
    u32 error;                 // sticky NECSIM_ERR_* (positive value of the negative code)
    u32 j_max;                 // largest event ordinal seen in a speciation record
    u32 n_unfinished;
    u32 n_sampled;             // written by the init kernels
    u32 n_rec;                 // event-stream records written this epoch (NEXT-3)
    u32 n_long;                // long runs of equal key prefix queued for stream_long_runs_kernel (NEXT-3)
    u32 pad_;
    u64 n_events;              // events executed (raw)
    u64 n_culled;
    u64 resamples;
    u64 tail_rounds_exact;     // tail kernel, exponential sampler: search rounds done in exact arithmetic (the fast round's fall-back count)
};

// Per-lineage SoA outputs + queues + dedup cache (all inside the simulate workspace).
struct SimBuffers {
    uint4 *q_in;               // {id, loc, cell, steps}
    uint4 *q_out;
    u32 q_in_count;
    uint4 *cache;              // {loc, k, j, owner id}; 0xFF.. = empty
    u32 cache_mask;
    u32 *term_loc, *term_k, *term_j, *steps, *parent, *spec_ring;
    u64 *term_f;
    uint8_t *state;            // 0 active, 1 speciated, 2 culled, 3 stopped by max_steps
    // event-stream ring of one epoch (REC kernels): one 32-byte record per executed event, written with two 16-byte stores --
    // rec[2i] = {origin loc, k, j, parent loc (0xFFFFFFFF = speciation)}, rec[2i+1] = {f lo, f hi, 0, 0} -- and its 64-bit time key
    // rec_key[i] = (k - k_start) << 40 | f >> 8, which the per-epoch sort works on (coalesced (key, index) pairs, no gathers)
    uint4 *rec;
    u64 *rec_key;
    u32 key_shift;             // 0: 64-bit keys; else the ring holds 32-bit keys (u32)(key >> key_shift) (the compact sort of an epoch of few intervals)
    u32 rec_cap;
    u32 k_base;                // radix passes sort k - k_base (0 for the species table; the epoch's k_start for the stream ring)
    SimCounters *ctr;
};

struct EpochArgs {
    SeedKey key;
    u64 thr_nu, thr_m;
    u32 k_start;               // every queued lineage is fresh at the start of interval k_start
    u32 k_stop;                // horizon: a lineage pauses when its interval index reaches k_stop
    u32 max_steps;             // 0 = unlimited
    u32 lanes_per_warp;        // lanes of each warp that hold lineages (32 = saturated; fewer in the tail)
    u32 rec_chunk;             // event-stream ring slots a tail-kernel warp reserves at a time (1..64)
    u32 probe_mask;            // an event probes the dedup cache iff hash & probe_mask == 0: the top log2(period) bits of the hash (0 = every event)
    u32 zero;                  // always 0, but only the host knows: ties instruction chains together in issue order (tail kernel)
};

}  // namespace necsim
