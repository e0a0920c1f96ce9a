/*
 * necsim.h -- C-ABI of libnecsim_b200.so: the Independent algorithm for individual-based neutral
 * (Moran) biodiversity simulation on one NVIDIA B200 (sm_100a).
 *
 * Paper: arxiv 2108.05815 (M. Langenstein, "Communication-free and Parallel Simulation of Neutral
 * Biodiversity Models"); "PAPER.md Lnnn" = line of /root/reference/PAPER.md. The arithmetic every
 * entry point performs is fixed by DESIGN.md section 2 (the paper leaves hash, logarithm and table
 * construction open; DESIGN.md section 3 lists those readings).
 *
 * Conventions
 *   - Every pointer argument says HOST or DEVICE. The library never allocates device memory: all
 *     device storage is a caller-provided workspace (size from the *_workspace_size queries, 256-byte
 *     aligned), e.g. a torch uint8 tensor. `cuda_stream` is a cudaStream_t passed as void* (NULL = the
 *     legacy default stream). All work is enqueued on that stream.
 *   - Return value: NECSIM_OK (0) or a negative NECSIM_ERR_* code; necsim_last_error() then returns a
 *     thread-local human-readable message. No exception or abort crosses this boundary.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns
 *     NECSIM_ERR_CUDA.
 */
#ifndef NECSIM_H
#define NECSIM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NECSIM_OK 0
#define NECSIM_ERR_INVALID_ARG (-1)
#define NECSIM_ERR_WORKSPACE_TOO_SMALL (-2)
#define NECSIM_ERR_CAPACITY (-3) /* k overflowed 2^32, resampling exhausted, too many epochs */
#define NECSIM_ERR_CUDA (-4)
#define NECSIM_ERR_UNSUPPORTED (-5)

/* Scenario kinds (PAPER.md 2.4, L284-302). */
#define NECSIM_NONSPATIAL 0
#define NECSIM_SPATIALLY_IMPLICIT 1
#define NECSIM_EXPLICIT_MATRIX 2
#define NECSIM_EXPLICIT_GAUSSIAN 3

/*
 * Scenario = habitat + turnover + dispersal (+ community sizes).
 * All arrays are HOST pointers, read during necsim_create_scenario only (the caller may free them
 * afterwards). Cells are row-major (cell = y*width + x) on a torus.
 */
typedef struct necsim_scenario_desc {
    int32_t kind;             /* NECSIM_NONSPATIAL .. NECSIM_EXPLICIT_GAUSSIAN */
    uint32_t width, height;   /* NONSPATIAL: 1x1. SPATIALLY_IMPLICIT: ignored */
    uint32_t sampler;         /* event-time sampler: 0 = exponential, 1 = Poisson / order
                                 statistics (L733-741). Same law, different realisation */
    const uint32_t *deme;     /* HOST [width*height] deme size per cell, 0 = not habitat; NULL = uniform_deme */
    uint32_t uniform_deme;
    const double *turnover;   /* HOST [width*height] lambda per cell (> 0, finite; read for habitat cells); NULL = uniform */
    double uniform_turnover;
    const double *dispersal_matrix; /* EXPLICIT_MATRIX: HOST [ncells*ncells] row-major, row = current cell,
                                       column = parent cell; >= 0, row sum > 0, 0 into non-habitat columns */
    double sigma;             /* EXPLICIT_GAUSSIAN: std-dev of the rounded normal displacement, in cells */
    uint64_t local_size;      /* SPATIALLY_IMPLICIT: J_local (sampleable) */
    uint64_t meta_size;       /* SPATIALLY_IMPLICIT: J_meta */
    double migration;         /* SPATIALLY_IMPLICIT: m in [0,1] */
    double delta_t;           /* repriming interval; 1/256 < lambda*delta_t <= 64 */
    /* Temporally varying habitat, EXPLICIT_GAUSSIAN only. `deme` is the present (era 0);
     * past_deme[e-1] (HOST [n_past_eras][width*height], n_past_eras <= 3) is the deme map of era e >= 1, in force for interval
     * indices k >= past_start_k[e-1] (HOST [n_past_eras], strictly increasing, > 0). Habitat is only lost towards the present:
     * every era's map contains the younger one cell by cell, else NECSIM_ERR_INVALID_ARG. Indexed locations (in events and the
     * event stream) are then canonical on the OLDEST map; the sample mask ranges over the present-day individuals. 0 = static. */
    uint32_t n_past_eras;
    const uint32_t *past_deme;
    const uint32_t *past_start_k;
} necsim_scenario_desc;

/*
 * Launch / scheduling knobs. NONE of them may change d_events, d_labels or richness: that is the
 * paper's reproducibility claim and tests/test_gpu_invariance.py checks it.
 * A zero field means "library default".
 */
typedef struct necsim_sim_params {
    uint32_t block_threads;    /* threads per block of the simulate kernels (multiple of 32, <= 256; default 256) */
    uint32_t grid_blocks;      /* persistent blocks; 0 = resident blocks per SM x number of SMs */
    uint32_t dedup;            /* 0 = default (on), 1 = on, 2 = off */
    uint32_t dedup_log2_slots; /* global duplicate-culling cache: 2^this slots of 16 bytes (default 22) */
    uint64_t epoch_events;     /* target number of events per epoch (time-horizon step, G.1 L2157-2187); 0 = default policy:
                                  half the cache slots and never fewer than 64 events per active lineage; the tail kernel runs as
                                  one launch without a horizon (with record_events: x64 per epoch, capped by the ring) */
    uint64_t max_steps;        /* 0 = unlimited; else a lineage stops after this many executed events
                                  ("unfinished": label 0xFFFFFFFF) -- the MODE-T throughput workload. With the duplicate
                                  culling on, WHICH lineages reach the cap depends on the launch shape (the cache is lossy: a
                                  lineage the oracle culls at its first shared event may run on here and hit the cap first), so
                                  only the labels of lineages with state 1 are reproducible then; with dedup = 2 (off) every
                                  per-lineage record is (tests/test_gpu_parity.py) */
    uint32_t tail_threshold;   /* switch to the low-latency tail kernel (one lineage per warp) when active lineages <= this;
                                  0 = default (128 lineages per SM) */
    uint32_t dedup_probe;      /* 0 = default: every 8th event probes the cache, every 32nd in the tail launch (a nested subset); else
                                  1 + log2 of the probe period for both kernels, 1..7: 1 = every event, 2 = every 2nd, ... 7 = every
                                  64th (chosen by a hash of the event identity; the paper probes every step_slice
                                  steps). Results never depend on it. */
    uint32_t record_events;    /* 1 = also produce the full event stream (PAPER.md 6.2 L813-906, 7.1.3 L958-967):
                                  every distinct executed event (speciation and dispersal), sorted by (k, f, loc, j) */
    uint32_t stream_sort_bytes;/* record_events: the radix sort of an epoch's records covers k and the leading 1..5 bytes of f; records
                                  that agree there are ordered by insertion (few, unless this is small). 0 = default: per epoch, the fewest
                                  bytes that leave about two records or fewer per value of that prefix. The
                                  stream does not depend on it */
    uint64_t event_ring_capacity;   /* records one epoch may produce (incl. redundant ones); 0 = 2^24. Each takes 60 bytes of workspace */
    uint64_t event_stream_capacity; /* distinct events of the whole run; 0 = 2^26. Each takes 24 bytes of workspace */
} necsim_sim_params;

/* One distinct speciation event = one species. 32 bytes. */
typedef struct necsim_event {
    uint32_t loc;       /* indexed location (x,y,i) as canonical linear id */
    uint32_t k;         /* repriming interval index */
    uint32_t j;         /* ordinal of the event inside interval k of loc's stream (>= 1) */
    uint32_t abundance; /* number of sampled individuals carrying this label */
    uint64_t f;         /* offset inside the interval, Q16.48, units of delta_t */
    double time;        /* ((double)k + f*2^-48) * delta_t, generations before present */
} necsim_event;

typedef struct necsim_result {
    /* compared bit-exactly with the oracle */
    uint64_t richness;            /* number of distinct speciation events reached */
    uint64_t n_lineages;          /* sampled individuals */
    uint64_t n_unfinished;        /* lineages stopped by max_steps */
    const necsim_event *d_events; /* DEVICE, inside the workspace: [richness], sorted by (k, f, loc, j) */
    const uint32_t *d_labels;     /* DEVICE: [n_lineages] index into d_events (sample order = ascending loc) */
    /* per-lineage terminal record (own path only): where it speciated / was culled / was stopped */
    const uint32_t *d_term_loc, *d_term_k, *d_term_j, *d_steps; /* DEVICE [n_lineages] */
    const uint64_t *d_term_f;                                   /* DEVICE [n_lineages] */
    const uint8_t *d_state;       /* DEVICE [n_lineages]: 1 speciated, 2 culled (duplicate), 3 stopped by max_steps */
    /* scheduling-dependent counters: reported, never compared (R20) */
    uint64_t n_events_raw;        /* events executed by all threads, including redundant ones */
    uint64_t n_culled;            /* lineages removed by the duplicate-culling cache */
    uint64_t n_speciation_raw;    /* speciation records before unique */
    uint64_t n_epochs;            /* simulate-kernel launches */
    uint64_t n_tail_epochs;       /* of which with the low-latency tail kernel */
    uint64_t resample_attempts;   /* rejected dispersal targets */
    uint64_t n_events_tail;       /* events executed in tail epochs */
    float ms_simulate;            /* device time of the simulate kernels (all epochs), CUDA events */
    float ms_simulate_tail;       /* of which tail epochs */
    float ms_total;               /* device time of the whole call */
    uint32_t n_kernel_launches;   /* kernels this call launched (memsets and copies not counted) */
    /* full event stream (record_events = 1), DEVICE SoA inside the workspace, [n_stream_events], sorted by (k, f, loc, j):
     * origin location, interval, ordinal, offset, and the parent's location (0xFFFFFFFF = the event is a speciation) */
    const uint32_t *d_stream_loc, *d_stream_k, *d_stream_j, *d_stream_loc2;
    const uint64_t *d_stream_f;
    uint64_t n_stream_events;
    /* tail kernel (exponential sampler): search rounds done in exact arithmetic (a fast round that was not clean is redone so,
     * DESIGN.md section 5); compare with n_events_tail. Reported, never compared */
    uint64_t n_tail_rounds_exact;
} necsim_result;

typedef struct necsim_scenario necsim_scenario;

/* Bytes of device workspace necsim_create_scenario needs for `desc` (tables of DESIGN.md section 4). */
int necsim_scenario_workspace_size(const necsim_scenario_desc *desc /*HOST*/, size_t *device_bytes /*HOST out*/);

/*
 * Validates `desc`, builds the per-cell tables (deme, prefix sums, turnover scales; alias tables for
 * EXPLICIT_MATRIX, R18; rounded-normal thresholds for EXPLICIT_GAUSSIAN, R15) on the host and uploads
 * them into `d_workspace` (DEVICE, `bytes` long), which must outlive the handle. Synchronises the
 * stream before returning. *out = NULL on failure.
 */
int necsim_create_scenario(const necsim_scenario_desc *desc /*HOST*/, void *d_workspace /*DEVICE*/, size_t bytes,
                           void *cuda_stream, necsim_scenario **out /*HOST out*/);

/* Length of the sample-mask domain: individuals in canonical order (cells row-major, deme index
 * ascending; SPATIALLY_IMPLICIT: the local community only). */
int necsim_scenario_num_individuals(const necsim_scenario *scn, uint64_t *n_individuals /*HOST out*/);

/* Bytes of device workspace one necsim_simulate call needs for up to n_sampled lineages. */
int necsim_simulate_workspace_size(const necsim_scenario *scn, uint64_t n_sampled, const necsim_sim_params *params /*HOST, NULL=defaults*/,
                                   size_t *device_bytes /*HOST out*/);

/*
 * Runs the whole hot path: traces every sampled individual backwards in time until
 * it speciates (PAPER.md 5.2, L675-747), culls duplicates (7.1.1, L940-946), and reduces the
 * speciation events to species (7.1.3, L958-967).
 *   seed : primes the hash RNG (5.2.1, L693-707).
 *   nu   : speciation probability per event in [0,1] (SPATIALLY_IMPLICIT: the metacommunity's; the
 *          local community has nu = 0, L1830). nu = 0 requires max_steps > 0.
 *   d_sample_mask : DEVICE u8[n_individuals], non-zero = sampled; NULL = everyone.
 *   n_sampled_capacity : the number of lineages the workspace was sized for (necsim_simulate_workspace_size); the
 *          mask is counted on the device and more sampled individuals than that => NECSIM_ERR_WORKSPACE_TOO_SMALL.
 *   bytes : size of d_workspace, at least what necsim_simulate_workspace_size returned for the same params.
 * Asynchronous on the stream except for one small read-back per epoch; returns after the final
 * read-back. Pointers in *out point into d_workspace and stay valid until it is reused.
 * One call at a time per scenario handle: the handle owns the pinned read-back block and the timing events of a call
 * (concurrent simulations need one handle each; the scenario workspace may be shared, it is read-only after creation).
 */
int necsim_simulate(necsim_scenario *scn, uint64_t seed, double nu, const uint8_t *d_sample_mask /*DEVICE or NULL*/,
                    uint64_t n_sampled_capacity, const necsim_sim_params *params /*HOST or NULL*/, void *d_workspace /*DEVICE*/,
                    size_t bytes, void *cuda_stream, necsim_result *out /*HOST out*/);

/*
 * Same, end to end with HOST buffers: copies h_sample_mask (HOST, may be NULL) to the device, simulates,
 * and copies events and labels back. h_events: HOST [n_sampled_capacity] (first richness entries
 * written) or NULL; h_labels: HOST [n_sampled_capacity] or NULL.
 */
int necsim_simulate_host(necsim_scenario *scn, uint64_t seed, double nu, const uint8_t *h_sample_mask /*HOST or NULL*/,
                         uint64_t n_sampled_capacity, const necsim_sim_params *params, void *d_workspace /*DEVICE*/, size_t bytes,
                         void *cuda_stream, necsim_result *out, necsim_event *h_events /*HOST*/, uint32_t *h_labels /*HOST*/);

/*
 * Merge of the species tables of isolated partitions ("IsolatedIndividuals / IsolatedLandscape", replay
 * L2511-2532): lineages simulated separately (other GPUs, other calls, later additions, L1485) reach the same
 * speciation events where they coalesce, so the union of the partitions' tables, made unique, is the table of the whole
 * sample. d_events_in: DEVICE [n] concatenation of d_events arrays; d_events_out: DEVICE [n] capacity, receives the
 * merged table sorted by (k, f, loc, j) with abundances added up; d_map: DEVICE [n], rank in the merged table of every
 * input record (a partition's labels are translated by map[offset_of_partition + label]); *richness: HOST out.
 */
int necsim_merge_workspace_size(uint64_t n, size_t *device_bytes /*HOST out*/);
int necsim_merge_species(const necsim_event *d_events_in /*DEVICE*/, uint64_t n, void *d_workspace /*DEVICE*/, size_t bytes, void *cuda_stream,
                         necsim_event *d_events_out /*DEVICE*/, uint32_t *d_map /*DEVICE*/, uint64_t *richness /*HOST out*/);

/*
 * necsim_merge_species for callers that cannot allocate device memory or pass a workspace (code under CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc): same inputs, outputs and results, but the sort / unique scratch of the merge kernels is
 * a static device array inside the library, sized for at most NECSIM_MERGE_STATIC_MAX input records (about 2.1 MB, held by every GPU
 * that loads the library until the process exits). n > NECSIM_MERGE_STATIC_MAX returns NECSIM_ERR_CAPACITY and touches nothing.
 * The call allocates nothing (no cudaMalloc / cudaFree, no allocating library routine); like necsim_merge_species it synchronises the
 * stream before it returns (*richness is a host value). All calls on one device share the one array: calls that overlap on the GPU
 * (different streams, different host threads) race on it -- serialise them. Nothing in the array has to be cleared between calls.
 */
#define NECSIM_MERGE_STATIC_MAX 65536u
int necsim_merge_species_static(const necsim_event *d_events_in /*DEVICE*/, uint64_t n, void *cuda_stream,
                                necsim_event *d_events_out /*DEVICE [n]*/, uint32_t *d_map /*DEVICE [n]*/, uint64_t *richness /*HOST out*/);

/* Frees the host-side handle (NULL is a no-op). The device workspace belongs to the caller. */
int necsim_destroy(necsim_scenario *scn);

/* Thread-local message for the last non-zero return of this thread. */
const char *necsim_last_error(void);

/* ---- test-only exports: run one device primitive over arrays (all array pointers DEVICE) -------- */
/* lane: 0 time, 1 spec, 2 disp (attempt r[i]; r may be NULL = 0), 3 index, 4 migr, 5 the primed state s */
int necsim_debug_draw(uint64_t seed, int lane, const uint32_t *d_loc, const uint32_t *d_k, const uint32_t *d_j, const uint32_t *d_r,
                      uint64_t *d_out, uint64_t n, void *cuda_stream);
/* fixed-point -ln, DESIGN.md 2.3 (PAPER.md Eq. C.3) */
int necsim_debug_neglog(const uint64_t *d_x, uint64_t *d_out, uint64_t n, void *cuda_stream);
/* The tail kernel's fast round decides the comparisons of the event-time search in binary32 where the outcome is
 * certain and redoes the round in fixed point otherwise. For every draw d_x[i] and the turnover scale (Cm, sh):
 * d_approx[i] = the binary32 offset of the draw, d_exact[i] = the Q16.48 offset of 2.4; *d_margin = the margin the kernel uses for
 * this scale. tests/test_gpu_primitives.py checks |approx - exact| against it. All pointers DEVICE. */
int necsim_debug_approx_time(const uint64_t *d_x, uint32_t Cm, uint32_t sh, float *d_approx, uint64_t *d_exact, float *d_margin, uint64_t n,
                             void *cuda_stream);
/* event-time search, DESIGN.md 2.4. rc[i]: 0 found, -3 k overflow */
int necsim_debug_next_event(uint64_t seed, const uint32_t *d_loc, const uint32_t *d_k, const int64_t *d_f_last, const uint32_t *d_Cm,
                            const uint32_t *d_sh, uint32_t *d_k_out, uint32_t *d_j_out, uint64_t *d_T_out, int32_t *d_rc, uint64_t n,
                            void *cuda_stream);
/* one dispersal from d_loc[i] at event (d_k[i], d_j[i]), DESIGN.md 2.5 step 2 */
int necsim_debug_disperse(const necsim_scenario *scn, uint64_t seed, const uint32_t *d_loc, const uint32_t *d_k, const uint32_t *d_j,
                          uint32_t *d_loc_out, uint64_t n, void *cuda_stream);
/* copies the scenario's device tables back to HOST arrays (any may be NULL): alias thresholds/aliases
 * [ncells*ncells], rounded-normal thresholds [2R] (*R_out = R), per-cell turnover scale Cm/sh [ncells] */
int necsim_debug_tables(const necsim_scenario *scn, uint32_t *h_thresh, uint32_t *h_alias, uint32_t *h_gauss, int32_t *R_out,
                        uint32_t *h_Cm, uint32_t *h_sh, void *cuda_stream);
/* Poisson sampler: event-time search over arrays; d_cell[i] = cell of d_loc[i] (thinning threshold) */
int necsim_debug_next_event_poisson(const necsim_scenario *scn, uint64_t seed, const uint32_t *d_loc, const uint32_t *d_cell, const uint32_t *d_k,
                                    const int64_t *d_f_last, uint32_t *d_k_out, uint32_t *d_j_out, uint64_t *d_T_out, int32_t *d_rc, uint64_t n,
                                    void *cuda_stream);
/* copies the Poisson cdf thresholds PC[256] and the per-cell thinning thresholds [ncells] to HOST (any may be NULL) */
int necsim_debug_poisson_table(const necsim_scenario *scn, uint64_t *h_pc, uint32_t *h_thin, double *mu_max, void *cuda_stream);
/* random-gather peak micro-benchmark ("a measured L2 random-sector peak"): every thread of a full-occupancy grid reads 8 bytes
 * from loads_per_thread pseudo-random 32-byte sectors of the caller's table (DEVICE, table_bytes long: smaller than L2 = the L2
 * random-sector peak, much larger = the HBM random-sector peak). Returns sector bytes (32 per load) per second. d_sink: DEVICE, 4 bytes. */
int necsim_debug_gather_peak(const void *d_table /*DEVICE*/, uint64_t table_bytes, uint32_t loads_per_thread, uint32_t *d_sink /*DEVICE*/,
                             void *cuda_stream, double *sector_bytes_per_s /*HOST out*/, float *ms /*HOST out*/);
/* integer-pipe peak micro-benchmark: runs `iters` iterations of an unrolled chain of
 * independent IMAD.WIDE / LOP3 / SHF / IADD3 on every SM; kind 0 = mixed hash-like, 1 = IMAD only,
 * 2 = ALU (LOP3/SHF/IADD3) only. d_sink: DEVICE, 4 bytes of the caller (keeps the chains alive; never written in practice).
 * Returns thread-level integer instructions per second. */
int necsim_debug_int_peak(int kind, uint32_t iters, uint32_t *d_sink /*DEVICE*/, void *cuda_stream, double *thread_instr_per_s /*HOST out*/,
                          float *ms /*HOST out*/);

#ifdef __cplusplus
}
#endif
#endif /* NECSIM_H */
