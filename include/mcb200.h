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
#define MC_EINVAL (-1)   /* bad argument, non-finite input, d <= 0, R <= 0 or > 1e7, l_B < 0, max_disp < 0, R/d_min > 1e6 */
#define MC_EOVERLAP (-2) /* two ions overlap in the initial configuration                          */
#define MC_EOUTSIDE (-3) /* an ion sticks out of the cavity in the initial configuration           */
#define MC_ENOSPACE (-4) /* workspace too small                                                    */
#define MC_ECUDA (-5)    /* a CUDA runtime call failed, or no sm_100 device                        */
#define MC_ESTALL (-6)   /* a sweep stalled (a wait of the sweep kernel exceeded "stall_ms"): the state is  \
                            invalid and every later sweep is a no-op until mc_set_positions / mc_set_state;  \
                            reported by every call that synchronises                                        */

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
 * validate = 0 skips the O(N^2) overlap check and the energy (E_running = 0).
 * Accuracy contract: per-trial dE within 1e-10 of max(|dE|, M_i) (reading G13) for any geometry
 * with cavity_R <= 1e7 and cavity_R / d_min <= 1e6; the pair-distance form is chosen from
 * cavity_R / d_min and max_disp / d_min (option "form"). */
int mc_init(mc_handle** out, int64_t N, const double* pos_dev, const double* charges_dev,
            const double* diameters_dev, double cavity_R, double bjerrum_length, double max_disp,
            uint64_t seed, void* workspace_dev, size_t workspace_bytes, void* stream, int validate);

/* n full sequential sweeps (sweep indices s .. s+n-1), enqueued, no host sync: ONE cooperative launch of
 * k_sweep per 1024 sweeps, trial generation included (PAPER.md:85-91 launched one kernel per cycle).
 * mc_sweep(a); mc_sweep(b) is bit-identical to mc_sweep(a+b).   PAPER.md:43-73, Alg. 1-5. */
int mc_sweep(mc_handle* h, int64_t n);

/* The same n sweeps -- the same chain, bit for bit in the accept/reject sequence -- by the paper's COMPARISON
 * code, the "parallel reduction scheme" of PAPER.md:278-282: one kernel launch per trial (N per sweep), the
 * N-1 pair terms spread over blocks of 1024 threads, warp-shuffle reductions, atomic sub-totals, a counter of
 * completed blocks, the last block decides.  Exists to reproduce the paper's comparison (Fig. 8-10), not for
 * speed.  Enqueued, no host sync.  mc_sweep and mc_sweep_reduction may be mixed freely. */
int mc_sweep_reduction(mc_handle* h, int64_t n);

/* From-scratch total energy l_B sum_{i<j} q_i q_j / r_ij in k_B T (monitored
 * during warm-up).  Synchronises. */
int mc_energy(mc_handle* h, double* E_host);

/* Same energy, left in device memory (E_dev, one double); enqueued, no host sync. */
int mc_energy_dev(mc_handle* h, double* E_dev);

/* The same energy for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no handle, no workspace, and the call itself calls no cudaMalloc, cudaFree
 * or allocating library routine.  E_dev (device, one double) := bjerrum_length * sum_{i<j} q_i q_j / r_ij (PAPER.md:60-63
 * Eq. 2's pair term summed over all pairs; the energy that is monitored) of the N ions at pos_dev
 * ([3][N], device) with charges charges_dev ([N], device), on the CURRENT device, enqueued on `stream` (a cudaStream_t,
 * NULL = the default stream), no host sync.  Inputs are not validated.  The per-CTA partial sums go through a static
 * __device__ array of 264,192 bytes that every GPU loading this library holds until exit; it is sized for
 * N <= MC_NOALLOC_MAX_N, a larger N is refused with MC_ENOSPACE (use mc_init + mc_energy there).  All calls on a
 * device share that array: calls that may overlap on the GPU (different streams, or graphs replayed concurrently)
 * race on it -- serialise them.  Nothing in the array has to be cleared between calls (every partial a call reads it
 * has written first).  Agrees with mc_energy to rounding (<= 1e-9 relative; same decomposition, exact coordinate
 * differences throughout). */
#define MC_NOALLOC_MAX_N 131072
int mc_energy_noalloc(int64_t N, const double* pos_dev /* [3][N] */, const double* charges_dev /* [N] */,
                      double bjerrum_length, double* E_dev, void* stream);

/* Adds the current configuration's ordered-pair distance counts into caller-owned device
 * accumulators: hist_dev [2][2][nbins] and n_centres_dev [2] (uint64).  Species index 0 if
 * q > 0 else 1.  Centres are ions with |x_i| <= centre_rmax (bulk only); partners
 * are all j != i; bin = floor(r / bin_width) computed as floor(r * (1/bin_width)) with IEEE
 * sqrt; pairs with bin >= nbins are dropped.  g(r) of PAPER.md:364-376.  Enqueued, no sync. */
int mc_pair_hist(mc_handle* h, double bin_width, int nbins, double centre_rmax,
                 uint64_t* hist_dev, uint64_t* n_centres_dev);

/* Same n sweeps through HOST buffers (the end-to-end path): if pos_in_host != NULL it is
 * uploaded ([3][N]) and replaces the configuration -- as mc_set_positions does (from-scratch
 * energy, O(N^2/2)) if E_running_in == NULL, else with E_running := *E_running_in taken on trust
 * (a caller that feeds back the positions and the E_running it just downloaded pays no extra
 * pass).  After the sweeps positions ([3][N]) and stats are downloaded into pos_out_host /
 * stats_host (either may be NULL).  Host buffers should be pinned for the copies to be
 * asynchronous.  Synchronises. */
int mc_sweep_host(mc_handle* h, int64_t n, const double* pos_in_host, const double* E_running_in,
                  double* pos_out_host, mc_stats* stats_host);

/* ---- accessors for parity tests, near-tie re-sync and checkpoint/resume.  The state of a chain is
 * the particle array (it is downloaded for analysis), the sweep counter that keys
 * the random stream (reading G9) and the running energy that is monitored. ---- */
int mc_get_positions(mc_handle* h, double* pos_dev_out /* [3][N] */);          /* enqueued */
/* Replaces the configuration (not validated); E_running := from-scratch energy; clears a stall. Enqueued. */
int mc_set_positions(mc_handle* h, const double* pos_dev /* [3][N] */);
/* Checkpoint resume in one call: configuration (not validated), sweep index and running energy as
 * saved from mc_get_positions / mc_get_sweep_index / mc_get_stats; no O(N^2) pass; clears a stall. Enqueued. */
int mc_set_state(mc_handle* h, const double* pos_dev /* [3][N] */, uint64_t sweep_index, double E_running);
int mc_get_sweep_index(mc_handle* h, uint64_t* s_host);                         /* synchronises */
int mc_set_sweep_index(mc_handle* h, uint64_t s);                               /* enqueued */
/* Counters since mc_init and the running energy (energy monitored during warm-up;
 * vetoes are counted apart from energy rejections).  Synchronises. */
int mc_get_stats(mc_handle* h, mc_stats* stats_host);
/* Log of the last sweep (Alg. 4: one decision per particle): dE_dev [N] (k_B T;
 * unspecified for overlap-vetoed trials, reading G14) and flags_dev [N]: bit0 accept, bit1 overlap
 * veto, bit2 wall veto, bit3 near-tie.  Either may be NULL.  Enqueued. */
int mc_get_trial_log(mc_handle* h, double* dE_dev, uint8_t* flags_dev);
int mc_free(mc_handle* h);

const char* mc_last_error(void);

/* Diagnostics for the roofline: runs a register-resident DFMA loop on every SM for about
 * `millis` ms on the given stream and returns FP64 FMA warp-lane instructions per second
 * (thread-level DFMA/s).  Synchronises.  Not part of the hot path. */
int mc_measure_fp64_peak(void* stream, double millis, double* dfma_per_second_host);

/* Diagnostics for the roofline: mc_sweep(h, n) (1 <= n <= 1024: one launch of k_sweep, which advances the chain
 * exactly as mc_sweep does) with a CUDA event pair on the handle's stream around the launch; *ms_host = its
 * device time.  The launch covers n N(N-1) pair evaluations that count.  Synchronises. */
int mc_sweep_timed(mc_handle* h, int64_t n, double* ms_host);

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
 * exactly once per chunk, and that the urgent items' release units hand out every MID and FIX item exactly
 * once, in the order in which the chain releases them (for 4, 8 and 16 columns per FIX item).  out4_host = {items, violations, widest item in columns, urgent items}. */
int mc_plan_check(int64_t N, int rows_per_thread, int far_cols, int far_workers, int64_t* out4_host);

/* Diagnostics: copies the first n ints of the sweep kernel's scheduling state -- W = 256 + 4 (N / 256 + 1) live
 * words (ticket counters, progress counter, per-chunk completion counters; zero between sweeps) followed by W
 * words that hold their values at the end of the last completed sweep; n <= 2 W -- or, for n < 0, the
 * first -n 32-bit words of the diagnostic counters (-n <= 2080) -- to the host on a stream of its
 * own, without waiting for the handle's stream (usable while a sweep is running). */
int mc_debug_peek(mc_handle* h, int32_t* out_host, int n);

/* Options.  Every setting gives the same accept/reject sequence as the oracle; settings that change
 * the partition of a row's sum change dE by rounding only (the sums themselves do not depend on the
 * schedule).  Unknown keys and out-of-range values return MC_EINVAL.
 *   "prows"        1|2|3|4 rows per thread of the sweep kernel; chunk = 256 * prows rows
 *                          (default by N: 3 from 36864, 2 from 512, else 1)
 *   "far_cols"     8..65536, multiple of 8: target columns per FAR item (default by N: 64 below 36864, 128 below 53248,
 *                          256 below 114688, else 384)
 *   "pnear"        0..128  worker CTAs that serve only urgent and in-chunk items (default 4 from N = 36864, else 8)
 *   "wave"         0|1     round a chunk's FAR items to a multiple of the FAR workers (default 1)
 *   "form"         -1|0|1|2  pair-distance form (persist.cuh): -1 = by geometry (default): 0 GRAM if
 *                          cavity_R / d_min <= 128, else 1 DIFFW if max_disp / d_min <= 64, else 2 CANON;
 *                          a value below the automatic one is refused (it would break the dE bar) unless
 *                          debug = 1 (measurements of that error)
 *   "position_bits" 64|32  32: the paper's storage format (float4 positions): the current
 *                          configuration is rounded to FP32 values (E_running := its from-scratch energy) and
 *                          every later trial position is rounded to FP32 once more; all pair arithmetic stays
 *                          FP64.  A different (equally valid) chain; the oracle has the same switch
 *   "uniform_path" 0|1     allow the equal-diameter specialisation (default 1)
 *   "stall_ms"     0..3600000  watchdog limit per wait of the sweep kernel in ms (default 2000; 0 = none;
 *                          raise it under a profiler, a sanitizer or GPU time-slicing)
 *   "diag_split"   0|1|2|4|8  warps that share one 32 x 32 in-chunk unit of the sweep kernel, each taking a part of
 *                          its columns -- the multi-thread-per-particle scheme of PAPER.md:243-245 for systems too
 *                          small to fill the device (0 = by N: 4 up to 768 ions, 2 up to 6144, else 1)
 *   "fix_cols"     0|4|8|16 columns per urgent item over the chunk just finished (0 = by N: 16 from N = 53248, 8 from 36864, else 4:
 *                          where the chain paces the sweep, many short items finish sooner than few long ones)
 *   "max_ctas"     0..4096 upper limit on the CTAs of the sweep kernel (0 = two per SM, the default for large
 *                          systems; small systems synchronise faster on a smaller grid)
 *   "energy_rows"  4|6|8   rows per thread of the from-scratch energy kernel
 *   "hist_slices"  1..64   column slices of the pair-histogram kernel (default 32)
 *   "debug"        0|1     collect the counters of mc_debug_counters (default 0)
 *   "probe"        0|1|2   needs debug = 1.  1: the next sweeps run the worker loop alone over all columns
 *                          (throughput probe); their results are meaningless and the sweep index stands still.
 *                          2: the deciding warp never runs, so the next sweep stalls (tests MC_ESTALL)
 * mc_get_option reads a setting back ("form_auto": the form the geometry allows; "grid": CTAs of the
 * last k_sweep launch, 2 per SM). */
int mc_set_option(mc_handle* h, const char* key, int64_t value);
int mc_get_option(mc_handle* h, const char* key, int64_t* value_host);

/* Number of kernels this handle launched (or replayed through graphs) since mc_init. */
int mc_get_launch_count(mc_handle* h, uint64_t* n_host);

#ifdef __cplusplus
}
#endif
#endif /* MCB200_H */
