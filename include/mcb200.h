/* mcb200.h -- C ABI of libmcb200.so: exact sequential-order Metropolis sweeps of a
 * primitive-model electrolyte (charged hard spheres, bare 1/r Coulomb, hard-wall spherical
 * cavity) on one NVIDIA B200 (sm_100a).  Hot path of arXiv 1602.05716 ("Brush Metropolis").
 *
 * What a sweep is: PAPER.md:43-52 (Sec. 2: select / trial / accept, Eq. 1; sequential updating
 * scheme = particles 0..N-1 in ascending order, each tried exactly once) with the pair-energy
 * dependency of PAPER.md:60-73 (Eq. 2: partner j<i enters with its already-decided position
 * x'_j, partner j>i with its sweep-start position x_j).  Energies are exact (no truncation,
 * PAPER.md:13, 33), all energy arithmetic is FP64, a hard-core overlap is a
 * separate integer veto, the domain is a hard-wall sphere.
 * Readings of silent/garbled points (G1..G19) are listed in DESIGN.md.
 *
 * Conventions
 *  - Plain C symbols, no C++/torch types.  Every function returns int: 0 = MC_OK, negative =
 *    error; it never throws and never exits.  mc_last_error() gives a message for the last
 *    failure on the calling thread.
 *  - "dev" pointers are CUDA device pointers on the current device, "host" pointers are host
 *    memory.  The library allocates NO device memory: the caller owns every buffer; the
 *    workspace is borrowed until mc_free().  Input arrays passed to mc_init are copied.
 *  - All work is enqueued on the stream given to mc_init (a cudaStream_t passed as void*, NULL
 *    = legacy default stream) and is asynchronous, except calls that return host scalars or
 *    fill host buffers, which synchronise that stream.
 *  - One handle = one Markov chain; a handle is not thread-safe.
 *  - Units: lengths in sigma, energies in k_B T (beta = 1).  Positions are SoA [3][N]
 *    (all x, then all y, then all z), FP64.
 */
#ifndef MCB200_H
#define MCB200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MC_OK 0
#define MC_EINVAL (-1)   /* bad argument, non-finite input, d <= 0, R <= 0, l_B < 0, max_disp < 0, R/d_min > 2e4 */
#define MC_EOVERLAP (-2) /* two ions overlap in the initial configuration                          */
#define MC_EOUTSIDE (-3) /* an ion sticks out of the cavity in the initial configuration           */
#define MC_ENOSPACE (-4) /* workspace too small                                                    */
#define MC_ECUDA (-5)    /* a CUDA runtime call failed, or no sm_100 device                        */
#define MC_ESTALL (-6)   /* the sweep kernel's watchdog fired (a wait exceeded 2 s): state invalid  */

typedef struct mc_handle mc_handle;

typedef struct mc_stats {
    uint64_t accepted;     /* accepted trials since mc_init                                  */
    uint64_t veto_overlap; /* trials vetoed by a hard-core overlap            */
    uint64_t veto_wall;    /* trials vetoed by the hard wall                  */
    uint64_t near_ties;    /* non-vetoed trials with |dE + ln u| < 1e-8 (may go either way)  */
    double E_running;      /* energy at init (or last mc_set_positions) + sum of accepted dE */
} mc_stats;

/* Bytes of device scratch mc_init needs for N ions (0 if N < 1). */
size_t mc_workspace_bytes(int64_t N);

/* Create a chain.  PAPER.md:83-87 (state = the particle array), 351 (hard-wall sphere).
 *   pos_dev [3][N], charges_dev [N] (valences, FP64), diameters_dev [N]: device, read once.
 *   cavity_R: wall radius; ion i is confined to |x_i| <= R - d_i/2 (touching allowed).
 *   bjerrum_length: l_B; pair energy = l_B q_i q_j / r in k_B T.
 *   max_disp: each trial component is uniform in (x - max_disp, x + max_disp)   (PAPER.md:351,
 *             Alg. 1 PAPER.md:129-135 with D = 2 max_disp and the old position added).
 *   seed: Philox4x32-10 key; counter = (particle, sweep_lo, sweep_hi, 0|1).
 *   workspace_dev/workspace_bytes: >= mc_workspace_bytes(N), 256-byte aligned.
 * Validates on the device (finite, d > 0, inside the wall, no overlapping pair: O(N^2)),
 * sets sweep index 0, E_running = from-scratch energy, counters 0.  Synchronises.
 * validate = 0 skips the O(N^2) overlap check and the energy (E_running = 0). */
int mc_init(mc_handle** out, int64_t N, const double* pos_dev, const double* charges_dev,
            const double* diameters_dev, double cavity_R, double bjerrum_length, double max_disp,
            uint64_t seed, void* workspace_dev, size_t workspace_bytes, void* stream, int validate);

/* n full sequential sweeps (sweep indices s .. s+n-1), enqueued, no host sync.
 * mc_sweep(a); mc_sweep(b) is bit-identical to mc_sweep(a+b).   PAPER.md:43-73, Alg. 1-5. */
int mc_sweep(mc_handle* h, int64_t n);

/* From-scratch total energy l_B sum_{i<j} q_i q_j / r_ij in k_B T (monitored
 * during warm-up).  Synchronises. */
int mc_energy(mc_handle* h, double* E_host);

/* Same energy, left in device memory (E_dev, one double); enqueued, no host sync. */
int mc_energy_dev(mc_handle* h, double* E_dev);

/* Adds the current configuration's ordered-pair distance counts into caller-owned device
 * accumulators: hist_dev [2][2][nbins] and n_centres_dev [2] (uint64).  Species index 0 if
 * q > 0 else 1.  Centres are ions with |x_i| <= centre_rmax (bulk only); partners
 * are all j != i; bin = floor(r / bin_width) computed as floor(r * (1/bin_width)) with IEEE
 * sqrt; pairs with bin >= nbins are dropped.  g(r) of PAPER.md:364-376.  Enqueued, no sync. */
int mc_pair_hist(mc_handle* h, double bin_width, int nbins, double centre_rmax,
                 uint64_t* hist_dev, uint64_t* n_centres_dev);

/* Same n sweeps through HOST buffers (the end-to-end path): if pos_in_host != NULL it is
 * uploaded ([3][N]) and replaces the configuration as mc_set_positions does; after the sweeps
 * positions ([3][N]) and stats are downloaded into pos_out_host / stats_host (either may be
 * NULL).  Host buffers should be pinned for the copies to be asynchronous.  Synchronises. */
int mc_sweep_host(mc_handle* h, int64_t n, const double* pos_in_host, double* pos_out_host,
                  mc_stats* stats_host);

/* ---- accessors for parity tests, near-tie re-sync and checkpoint/resume ---- */
int mc_get_positions(mc_handle* h, double* pos_dev_out /* [3][N] */);          /* enqueued */
/* Replaces the configuration (not validated); E_running := from-scratch energy. Enqueued. */
int mc_set_positions(mc_handle* h, const double* pos_dev /* [3][N] */);
int mc_get_sweep_index(mc_handle* h, uint64_t* s_host);                         /* synchronises */
int mc_set_sweep_index(mc_handle* h, uint64_t s);                               /* enqueued */
int mc_get_stats(mc_handle* h, mc_stats* stats_host);                           /* synchronises */
/* Log of the last sweep: dE_dev [N] (k_B T; unspecified for overlap-vetoed trials) and
 * flags_dev [N]: bit0 accept, bit1 overlap veto, bit2 wall veto, bit3 near-tie.  Enqueued. */
int mc_get_trial_log(mc_handle* h, double* dE_dev, uint8_t* flags_dev);
int mc_free(mc_handle* h);

const char* mc_last_error(void);

/* Diagnostics for the roofline: runs a register-resident DFMA loop on every SM for about
 * `millis` ms on the given stream and returns FP64 FMA warp-lane instructions per second
 * (thread-level DFMA/s).  Synchronises.  Not part of the hot path. */
int mc_measure_fp64_peak(void* stream, double millis, double* dfma_per_second_host);

/* Diagnostics for the roofline: runs ONE sweep (it advances the chain exactly as mc_sweep(h, 1)
 * does, same kernels, same arguments, bit-identical result) with the kernels launched one after
 * the other on the handle's stream and a CUDA event pair around every launch.  Fills
 * ms_host[MC_NKERNELS] with the summed device time per kernel class and launches_host[MC_NKERNELS]
 * with the launch counts, pairs_host[MC_NKERNELS] with the pair evaluations (counted towards
 * N(N-1): rows x columns, no speculative work) each class covered.  Synchronises. */
#define MC_K_TRIAL 0
#define MC_K_BULK 1   /* rows of a chunk x columns outside chunks c-1, c                  */
#define MC_K_FIX 2    /* rows of a chunk x columns of chunk c-1 (same kernel as MC_K_BULK) */
#define MC_K_DIAG 3   /* rows of a chunk x columns of the chunk, with speculation          */
#define MC_K_CHAIN 4  /* sequential resolution                                             */
#define MC_NKERNELS 5
int mc_sweep_timed(mc_handle* h, double* ms_host, int64_t* launches_host, int64_t* pairs_host);

/* Diagnostics of the persistent sweep kernel (option "debug" = 1): SM-clock cycle counters of the
 * last sweep, out16_host[16]: [0] chain warp, whole sweep; [1] of which waiting for the first tile
 * of a chunk; [2] waiting for later tiles; [3] helper 0 waiting for FAR/DIAG of a chunk; [4] for
 * FIX; [5] summed cycles worker CTAs spent fetching items; [6..9] number of exit/DIAG/FAR/FIX
 * items fetched.  Synchronises. */
int mc_debug_counters(mc_handle* h, int64_t* out16_host);

/* Host-only check of the persistent kernel's work decomposition (no GPU needed): enumerates, for every
 * chunk of 256 * rows_per_thread rows of an N-particle system, the FAR-L, FAR-U, MID, FIX and DIAG
 * items exactly as the kernel slices them (far_cols = target columns per FAR item, far_workers = the
 * number the item counts are rounded to, 0 = no rounding) and verifies that every column is covered
 * exactly once per chunk.  out4_host = {items, violations, widest item in columns, urgent items}. */
int mc_plan_check(int64_t N, int rows_per_thread, int far_cols, int far_workers, int64_t* out4_host);

/* Diagnostics: copies the first n ints of the persistent kernel's scheduling state (ticket
 * counters, progress counter, per-chunk completion counters) to the host on a stream of its own,
 * without waiting for the handle's stream (usable while a sweep is running). */
int mc_debug_peek(mc_handle* h, int32_t* out_host, int n);

/* Tuning knobs (diagnostic; defaults are right for B200): key "chunk" = rows resolved per
 * chain kernel (multiple of 32, 32..1024), "graph" = 0/1 use CUDA graphs, "overlap" = 0/1 run
 * the chain concurrently with the next chunk's bulk kernel, "bulk_rows" = 1|2 rows per thread of
 * the bulk kernel, "bulk_ctas" = 1..4 bulk CTAs per SM the grid is sized for, "uniform_path" =
 * 0/1 allow the equal-diameter specialisation.  Every setting gives the same accept/reject
 * sequence; settings that change the partition of a row's sum change dE by rounding only.
 * Returns MC_EINVAL for unknown keys. */
int mc_set_option(mc_handle* h, const char* key, int64_t value);

/* Number of kernels this handle launched (or replayed through graphs) since mc_init. */
int mc_get_launch_count(mc_handle* h, uint64_t* n_host);

#ifdef __cplusplus
}
#endif
#endif /* MCB200_H */
