// persist.cuh -- one persistent kernel per sweep (sm_100a).  See DESIGN.md section 6.
//
// grid = 2 CTAs per SM, all co-resident (cooperative launch).  CTA 0 is the chain: it resolves the
// sweep's N decisions in ascending order.  Every other CTA is a worker that
// pulls items from three queues (ticket counters in global memory):
//   DIAG(c)  speculative corrections inside chunk c (in-chunk units)                        (a2/a3)
//   FAR(c)   rows of chunk c x a slice of the columns outside chunks c-1 and c          (a2)
//            DIAG and FAR of chunk c are released when the chain has finished chunk c-2
//   FIX(c)   rows of chunk c x 16 columns of chunk c-1 at their final positions         (a2)
//            urgent: exists as soon as the chain has published those columns' row group
// Every item adds its rows' partial sums into per-row 64-bit fixed-point accumulators with integer
// atomics (accum_row): integer addition is associative, so the sums -- and with them every accept
// bit -- do not depend on which CTA ran which item or in what order.
// The chain CTA: warp 0 decides (one ballot per step, Alg. 4); warps 1..6 each
// own row tiles t = w-1 (mod 6): they read the tile's base sum, add the corrections of all column
// tiles s <= t-2 as their accept masks appear, and hand the tile over through shared memory with
// the two blocks D(t,t-1), D(t,t) the chain warp applies itself (one bulk copy); warp 7 commits
// the accepted moves, writes the trial log and publishes progress to the workers.
#pragma once
#include "kernels.cuh"

namespace mcb {

constexpr int kPThreads = kBulkThreads;        // workers: 8 consumer warps; thread 0 also feeds the column ring
#ifndef MCB_GROUP
#define MCB_GROUP 128
#endif
#ifndef MCB_FIXCOLS
#define MCB_FIXCOLS 16
#endif
#ifndef MCB_MIDCOLS
#define MCB_MIDCOLS 32
#endif
constexpr int kGroup = MCB_GROUP;              // rows per published progress step of the chain
constexpr int kFixCols = MCB_FIXCOLS;          // columns per FIX item (columns of chunk c-1): the default for large systems;
                                               // PArgs::fixcols is what a launch uses (4 where the chain paces the sweep)
constexpr int kMidCols = MCB_MIDCOLS;          // columns per MID item (columns of chunk c-2)
#ifndef MCB_RING
#define MCB_RING 3
#endif
constexpr int kRing = MCB_RING;                // hand-off ring depth of the chain CTA (measured: 3 beats 4 and 2 at every N)
constexpr int kHelpers = 6;
#ifndef MCB_DRING
#define MCB_DRING 4
#endif
constexpr int kDRing = MCB_DRING;                      // D / overlap-bit buffers: DIAG(c) may run once the chain has finished chunk c - kDRing
#ifndef MCB_COLS_PER_ITER
#define MCB_COLS_PER_ITER 4
#endif
constexpr int kColsPerIter = MCB_COLS_PER_ITER;   // columns per iteration of the pair loop (2 pairs of rows x columns in flight per row)

// scheduling state in global memory; zero at the start of every sweep (cleared by CTA 0 at the end of the one before)
// (hot words 128 bytes apart, so that polling one does not slow down atomics on another)
enum { kSyTicket = 0, kSyUTicket = 32, kSyGroups = 64, kSyChainSm = 96, kSyDTicket = 128, kSyAbort = 160, kSyTicketU = 192,
       kSyHdr = 256 };

struct PArgs {
    Params p;
    int C;            // rows per chunk = 256 * ROWS
    int nchunks;
    int farcols;      // target columns per FAR item (multiple of 8)
    int nnear;        // worker CTAs 1..nnear serve FIX and DIAG only
    int nfar;         // number of FAR workers (0: do not round item counts to it)
    int mode;         // 0 normal; 1 throughput probe: no chain, every CTA runs QU items over all columns but the chunk's own;
                      // 2 watchdog test: the deciding warp never runs, so the sweep stalls
    int dsplit;       // warps that share one DIAG unit: 1, 2, 4 or 8
    int fixcols;      // columns per FIX item: 4, 8 or 16
    int nsweeps;      // sweeps this launch runs (a1-a4 each), separated by grid-wide barriers
    int* sy;          // [kSyHdr + 3 * nchunks]: header, far_done, diag_done, fix_done; all zero at launch and again at exit
    int* gbar;        // grid barrier: [0] arrivals, [32] generation
    long long* dbg;   // [16] diagnostic cycle counters (see mc_debug_counters), may be null
    int* uc;          // claim counters of the urgent release units (urgent_units() ints, zero between sweeps), see fetch_item
};

__host__ __device__ inline int chunk_rows(int Np, int C, int c) { return min(C, Np - c * C); }
// FAR items of one chunk over ncols columns: about farcols columns each, and -- when there are at
// least half as many as FAR workers -- a whole number of items per worker, so that a wave of items
// ends for all workers at about the same time
__host__ __device__ inline int far_slices(int ncols, int farcols, int nfar) {
    int n = (ncols + farcols - 1) / farcols;
    if (nfar > 0 && 2 * n >= nfar) n = ((2 * n + nfar) / (2 * nfar)) * nfar;   // nearest multiple, at least one
    if (n > ncols / 8) n = ncols / 8;
    return n;
}
// columns of the FAR items of chunk c: L = before chunk c-2 (final positions once the chain has
// finished chunk c-3), U = after chunk c (sweep-start positions, never blocked)
__host__ __device__ inline int farL_cols(int C, int c) { return c >= 3 ? (c - 2) * C : 0; }
// urgent items of chunk c: MID (columns of chunk c-2, c >= 2) then FIX (columns of chunk c-1, c >= 1)
__host__ __device__ inline int urgent_items(int C, int c, int fixcols = kFixCols) {
    return (c >= 2 ? C / kMidCols : 0) + (c >= 1 ? C / fixcols : 0);
}
// The urgent items are claimed by RELEASE UNIT: all items of a unit become claimable at the same moment -- MID(c), the
// C / kMidCols items over the columns of chunk c-2, when the chain has finished chunk c-2; FIX(c, g), the
// kGroup / kFixCols items over group g of chunk c-1, when the chain has published that group -- so one atomicAdd on the
// unit's counter hands out its items in parallel and can never reach into work that does not exist yet.  (Round 1 and
// the first half of round 2 took urgent tickets in order with a compare-and-swap: the eight items of a group were
// claimed one round trip after the other, 3.5 us for the last one at every chunk boundary.)
// Units in release order: chunk 1: FIX groups 0..GPC-1;  chunk c >= 2: MID(c), then FIX groups 0..GPC-1.
__host__ __device__ inline int urgent_units(int C, int nchunks) {
    const int GPC = C / kGroup;
    return nchunks >= 2 ? GPC + (nchunks - 2) * (GPC + 1) : 0;
}
__host__ __device__ inline int farU_cols(int Np, int C, int c) { return Np - (c * C + chunk_rows(Np, C, c)); }
__host__ __device__ inline int probe_cols(int Np, int C, int c) { return Np - chunk_rows(Np, C, c); }
__host__ __device__ inline int far_items(int Np, int C, int farcols, int nfar, int c) {
    return far_slices(farL_cols(C, c), farcols, nfar) + far_slices(farU_cols(Np, C, c), farcols, nfar);
}
// DIAG items of a chunk: nt x nt units of 32 x 32, each shared by `split` warps (1, 2, 4 or 8), 8 warps per item
__host__ __device__ inline int diag_items(int nrows, int split) {
    const int nt = nrows / kTile;
    return (nt * nt * split + 7) / 8;
}

__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ double2 ldcg2(const double2* p) {
    double2 v;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
// Watchdog: no wait in this kernel may last longer than Params::wait_limit_ns (option "stall_ms",
// default 2 s; 0 = no limit).  A thread whose wait does raises the abort flag (and DevState::stall,
// which every synchronising call of the host reports as MC_ESTALL) and exits; every other waiting
// thread sees the flag and exits too, so a scheduling bug can never hang the GPU.
struct Watch {
    int* sy;
    DevState* st;
    unsigned long long limit;
};
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
static __device__ __noinline__ void wd_check(const Watch& w, unsigned long long t0) {
    if (*(volatile int*)(w.sy + kSyAbort) == 0) {
        if (w.limit == 0ull || global_ns() - t0 < w.limit) return;
        *(volatile int*)(w.sy + kSyAbort) = 1;
        *(volatile int*)(&w.st->stall) = 1;
        __threadfence();
    }
    asm volatile("exit;");
}
// the same test without the exit: true if the kernel is being abandoned (raises the flags itself when the limit has passed)
static __device__ __noinline__ bool wd_poll(const Watch& w, unsigned long long t0) {
    if (*(volatile int*)(w.sy + kSyAbort) != 0) return true;
    if (w.limit == 0ull || global_ns() - t0 < w.limit) return false;
    *(volatile int*)(w.sy + kSyAbort) = 1;
    *(volatile int*)(&w.st->stall) = 1;
    __threadfence();
    return true;
}
__device__ __forceinline__ void spin_until_ge(const Watch& w, const int* p, int v) {
    if (ld_acquire(p) >= v) return;
    const unsigned long long t0 = global_ns();
    for (unsigned it = 1; ld_acquire(p) < v; ++it) {
        __nanosleep(64);
        if ((it & 1023u) == 0u) wd_check(w, t0);
    }
}
__device__ __forceinline__ void mbar_wait_wd(const Watch& w, uint64_t* bar, uint32_t parity) {
    if (mbar_try_wait(bar, parity)) return;
    const unsigned long long t0 = global_ns();
    for (unsigned it = 1; !mbar_try_wait(bar, parity); ++it)
        if ((it & 4095u) == 0u) wd_check(w, t0);
}

// shared memory of one CTA: workers use the column ring, the chain CTA the hand-off ring
struct HandOff {
    double D[3 * kTile * kTile];   // blocks (t, t-2), (t, t-1) and (t, t), [jj][lane] each (contiguous in Dblk)
    double E[kTile], lbq[kTile], lnu[kTile];
    double2 txy[kTile];
    double tz[kTile];
    unsigned ovoP[kTile], ovnP[kTile], ovoD[kTile], ovnD[kTile];
    unsigned veto[kTile];
    double out_dE[kTile];          // written by the chain warp, read by the publisher
    unsigned out_flags[kTile];
};

struct __align__(128) PShared {
    union {
        struct {
            ColStage stage[kStages];
            double2 cxy[8][32], czq[8][32], ctxy[8][32];
            double ch[8][32], ctz[8][32];
            unsigned ov[8][2][32];
        } w;
        HandOff ho[kRing];
    } u;
    uint64_t full_bar[kStages], empty_bar[kStages];
    uint64_t ho_bar[kRing];               // tile handed over by its helper
    uint64_t d_bar[kRing];                // the tile's three D blocks have landed in the slot (bulk-copy bytes)
    uint64_t p_bar[kRing];                // publisher done with the slot
    uint64_t a_bar[2][kChunkMax / kTile]; // accept mask of tile t of a chunk (by chunk parity) published
    unsigned sA[2][kChunkMax / kTile];
    int pub_gt;       // chain CTA: 1 + the last tile the publisher has taken out of its slot (monotonic within a sweep)
    int item[4];      // [0] type, [1] chunk, [2] index, [3] CTA flags (bit 0 idle, bit 1 abandoned)
};

__device__ __forceinline__ int* sy_far_done(const PArgs& a) { return a.sy + kSyHdr; }
__device__ __forceinline__ int* sy_diag_done(const PArgs& a) { return a.sy + kSyHdr + a.nchunks; }
__device__ __forceinline__ int* sy_fix_done(const PArgs& a) { return a.sy + kSyHdr + 2 * a.nchunks; }

// per-chunk view of the scratch double-buffered by chunk parity
struct ChunkBufs {
    double* Dblk;                       // [nt (nt + 1) / 2][32][32]
    unsigned* OVold; unsigned* OVnew;   // [C][C / 32]
};
__device__ __forceinline__ ChunkBufs chunk_bufs(const PArgs& a, int c) {
    const size_t b = (size_t)(c % kDRing);
    const size_t nt = kChunkMax / kTile;
    ChunkBufs B;
    B.Dblk = a.p.Dblk + b * (nt * (nt + 1) / 2) * (kTile * kTile);
    B.OVold = a.p.OVold + b * kChunkMax * nt;
    B.OVnew = a.p.OVnew + b * kChunkMax * nt;
    return B;
}

}  // namespace mcb

namespace mcb {

// exact overlap re-check with L2 loads (columns may have been rewritten by the chain during this kernel)
static __device__ __noinline__ int recheck_overlap_cg(const double2* xy, const double2* zq, const double* hh, double2 t,
                                               double tz, double hi, int v0, int v1, int cbeg, int gapv, int gap) {
    int ov = 0;
    for (int v = v0; v < v1; ++v) {
        const int j = cbeg + (v < gapv ? v : v + gap);
        const double2 a = ldcg2(xy + j);
        const double zj = __ldcg(&zq[j].x);
        const double sij = __dadd_rn(hi, hh[j]);
        const double r2n = dist2(__dadd_rn(t.x, -a.x), __dadd_rn(t.y, -a.y), __dadd_rn(tz, -zj));
        ov |= (r2n < __dmul_rn(sij, sij)) ? 1 : 0;
    }
    return ov;
}

// Pair evaluation (Eq. 2; Alg. 2) in three forms, chosen by mc_init from the
// geometry so that the per-trial dE stays within 1e-10 of its natural scale:
//  GRAM  (20 FP64-pipe instructions + 2 MUFU; 22 if diameters differ)    cavity_R / d_min <= 128
//     r2o = |x_i|^2 + |x_j|^2 - 2 x_i.x_j       1 DADD + 3 DFMA   (|x_j|^2 is staged with the column)
//     w   = 2 D.x_i + |D|^2 - 2 D.x_j           3 DFMA            (D = x~_i - x_i)
//     r2n = r2o + w                             1 DADD
//     absolute error of r2o: a few ulp(R^2), i.e. <= 5e-15 (R/r)^2 relative in 1/r
//  DIFFW (22; 24)                                                         max_disp / d_min <= 64
//     dx = x_i - x_j ... (3 DADD), r2o = fma(dz,dz,fma(dy,dy,dx dx)) (3), w = 2 D.dx + |D|^2 (3), r2n = r2o + w (1)
//     r2o as the oracle forms it; r2n carries an absolute error of a few ulp((r_o + max_disp)^2)
//  CANON (25; 27: the canonical count of SURVEY.md 8(d))                  any geometry
//     both distances from rounded differences, exactly as reading G11 writes them
// plus, in every form, 2 x 5 for the rsqrt refinements and 2 for the difference and the accumulate.
// The overlap veto is an integer test off the FP64 pipe: a running signed minimum
// (VIMNMX3, one per two pairs) of the high word of r2n (equal diameters) or of r2n - s_ij^2.
// A negative r2n (possible in the GRAM form when the trial lands within ~1e-6 sigma of another centre) has a
// negative high word and so wins the minimum: it reads as an overlap, never as a large distance.
// A row whose minimum falls inside a narrow band around contact -- where the re-associated r2n could
// differ from reading G11's evaluation order -- is re-examined exactly (recheck_overlap_cg).
enum { kFormGram = 0, kFormDiffW = 1, kFormCanon = 2 };
constexpr int kOvBand = 16;   // equal diameters: band of +-16 high-word steps (2^-16 relative) around s^2

struct RowP {
    double a0, a1, a2;  // GRAM: -2 x_i            DIFFW, CANON: x_i
    double b0, b1, b2;  // GRAM: -2 D              DIFFW: 2 D            CANON: x~_i
    double c0;          // GRAM: |x_i|^2           DIFFW: |D|^2
    double c1;          // GRAM: 2 D.x_i + |D|^2
    double h;           // d/2
    double acc;
    int m;              // running minimum of the overlap key
};

template <int FORM>
__device__ __forceinline__ void row_init(RowP& r, double2 xyi, double zi, double2 txyi, double tzi, double ni, double hi) {
    const double Dx = __dadd_rn(txyi.x, -xyi.x), Dy = __dadd_rn(txyi.y, -xyi.y), Dz = __dadd_rn(tzi, -zi);
    if (FORM == kFormGram) {
        r.a0 = __dmul_rn(-2.0, xyi.x); r.a1 = __dmul_rn(-2.0, xyi.y); r.a2 = __dmul_rn(-2.0, zi);
        r.b0 = __dmul_rn(-2.0, Dx); r.b1 = __dmul_rn(-2.0, Dy); r.b2 = __dmul_rn(-2.0, Dz);
        r.c0 = ni;
        // 2 D.x_i + |D|^2 = D.(2 x_i + D)
        r.c1 = __fma_rn(Dx, __fma_rn(2.0, xyi.x, Dx), __fma_rn(Dy, __fma_rn(2.0, xyi.y, Dy), __dmul_rn(Dz, __fma_rn(2.0, zi, Dz))));
    } else if (FORM == kFormDiffW) {
        r.a0 = xyi.x; r.a1 = xyi.y; r.a2 = zi;
        r.b0 = __dadd_rn(Dx, Dx); r.b1 = __dadd_rn(Dy, Dy); r.b2 = __dadd_rn(Dz, Dz);
        r.c0 = dist2(Dx, Dy, Dz);
        r.c1 = 0.0;
    } else {
        r.a0 = xyi.x; r.a1 = xyi.y; r.a2 = zi;
        r.b0 = txyi.x; r.b1 = txyi.y; r.b2 = tzi;
        r.c0 = 0.0; r.c1 = 0.0;
    }
    r.h = hi;
    r.acc = 0.0;
    r.m = 0x7fffffff;
}

template <int FORM, bool UNIFORM>
__device__ __forceinline__ int pair_eval(RowP& r, const double2 a, const double2 b, double nj, double hj) {
    double r2o, r2n;
    if (FORM == kFormGram) {
        r2o = __fma_rn(r.a0, a.x, __fma_rn(r.a1, a.y, __fma_rn(r.a2, b.x, __dadd_rn(r.c0, nj))));
        const double w = __fma_rn(r.b0, a.x, __fma_rn(r.b1, a.y, __fma_rn(r.b2, b.x, r.c1)));
        r2n = __dadd_rn(r2o, w);
    } else {
        const double dx = __dadd_rn(r.a0, -a.x), dy = __dadd_rn(r.a1, -a.y), dz = __dadd_rn(r.a2, -b.x);
        r2o = dist2(dx, dy, dz);
        if (FORM == kFormDiffW) {
            const double w = __fma_rn(r.b0, dx, __fma_rn(r.b1, dy, __fma_rn(r.b2, dz, r.c0)));
            r2n = __dadd_rn(r2o, w);
        } else {
            r2n = dist2(__dadd_rn(r.b0, -a.x), __dadd_rn(r.b1, -a.y), __dadd_rn(r.b2, -b.x));
        }
    }
    int key;
    if (UNIFORM) {
        key = __double2hiint(r2n);
    } else {
        const double sij = __dadd_rn(r.h, hj);
        key = __double2hiint(__fma_rn(-sij, sij, r2n));   // sign and magnitude of r2n - s_ij^2
    }
    const double du = __dadd_rn(rsqrt_fast(r2n), -rsqrt_fast(r2o));
    r.acc = __fma_rn(b.y, du, r.acc);
    return key;
}

// What the running minimum m of a row's keys says about the veto: 1 overlap, 0 none, -1 inside the band
// (re-examine exactly).  Signed order of the high words: any negative value (r2n < 0, or r2n - s^2 < 0)
// is below every positive one, and among negative doubles the one closest to zero has the smallest word.
template <bool UNIFORM>
__device__ __forceinline__ int veto_from_min(int m, double h, double ov_tol) {
    if (UNIFORM) {
        if (m < 0) return 1;                                    // r2n itself came out negative: on top of a centre
        const double s = __dadd_rn(h, h);
        const int key = m - __double2hiint(__dmul_rn(s, s));     // both words in [0, 0x7ff00000): no wrap
        return key < -kOvBand ? 1 : key > kOvBand ? 0 : -1;
    }
    const int tolhi = __double2hiint(ov_tol);
    if (m >= tolhi) return 0;                                   // smallest r2n - s^2 is clearly positive
    if (m < 0 && (m & 0x7fffffff) >= tolhi) return 1;           // the negative one closest to zero is clearly negative
    return -1;
}

// FAR / FIX item: all rows of the chunk (ROWS per consumer thread) x virtual columns [v0, v1) of
// the column space that starts at cbeg and skips [gap0, gap1).  The
// mbarrier ring persists across items (kring = stages used so far, identical in every thread).
template <int ROWS, bool UNIFORM, int FORM>
__device__ __forceinline__ void bulk_item(const Params& p, PShared& sh, unsigned& kring, int row0, int nrows,
                                          int cbeg, int gap0, int gap1, int v0, int v1) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int gap = gap1 - gap0;
    const int gapv = gap0 - cbeg;
    const Watch wd{p.sy, p.st, p.wait_limit_ns};

    // producer state (thread 0 only): next stage to issue
    unsigned kp = kring;
    int vp = v0;
    auto issue = [&]() {
        const int lim = (vp < gapv) ? min(v1, gapv) : v1;
        const int cnt = min(kColTile, lim - vp);
        const int a = cbeg + ((vp < gapv) ? vp : vp + gap);
        const unsigned s = kp % kStages;
        if (kp >= (unsigned)kStages) mbar_wait_wd(wd, &sh.empty_bar[s], ((kp / kStages) - 1) & 1);
        mbar_arrive_expect_tx(&sh.full_bar[s], (uint32_t)cnt * (32u + (FORM == kFormGram ? 8u : 0u) + (UNIFORM ? 0u : 8u)));
        bulk_g2s(sh.u.w.stage[s].xy, p.xy + a, (uint32_t)cnt * 16u, &sh.full_bar[s]);
        bulk_g2s(sh.u.w.stage[s].zq, p.zq + a, (uint32_t)cnt * 16u, &sh.full_bar[s]);
        if (FORM == kFormGram) bulk_g2s(sh.u.w.stage[s].n, p.nn + a, (uint32_t)cnt * 8u, &sh.full_bar[s]);
        if (!UNIFORM) bulk_g2s(sh.u.w.stage[s].h, p.hh + a, (uint32_t)cnt * 8u, &sh.full_bar[s]);
        vp += cnt;
        ++kp;
    };
    if (tid == 0) {
        fence_proxy_async();
        for (int q = 0; q < kStages - 1 && vp < v1; ++q) issue();
    }

    RowP R[ROWS];
#pragma unroll
    for (int u = 0; u < ROWS; ++u) {
        const int r = u * kBulkThreads + tid;
        const int i = row0 + (r < nrows ? r : 0);
        const double2 xyi = ldcg2(p.xy + i);
        row_init<FORM>(R[u], xyi, __ldcg(&p.zq[i].x), p.txy[i], p.tz[i], FORM == kFormGram ? __ldcg(p.nn + i) : 0.0, p.hh[i]);
    }
    const bool warp_live = warp * 32 < nrows;

    unsigned k = kring;
    for (int v = v0; v < v1; ++k) {
        const int lim = (v < gapv) ? min(v1, gapv) : v1;
        const int cnt = min(kColTile, lim - v);
        const unsigned s = k % kStages;
        if (tid == 0 && vp < v1) issue();   // keeps kStages - 1 stages in flight ahead of this one
        __syncwarp();
        mbar_wait_wd(wd, &sh.full_bar[s], (k / kStages) & 1);
        const ColStage& st = sh.u.w.stage[s];
        if (warp_live) {
            auto cols = [&](int j0) {
#pragma unroll
                for (int jj = 0; jj < kColsPerIter; jj += 2) {
                    const double2 a0 = st.xy[j0 + jj], a1 = st.xy[j0 + jj + 1];
                    const double2 b0 = st.zq[j0 + jj], b1 = st.zq[j0 + jj + 1];
                    const double h0 = UNIFORM ? 0.0 : st.h[j0 + jj], h1 = UNIFORM ? 0.0 : st.h[j0 + jj + 1];
                    const double n0 = FORM == kFormGram ? st.n[j0 + jj] : 0.0, n1 = FORM == kFormGram ? st.n[j0 + jj + 1] : 0.0;
#pragma unroll
                    for (int u = 0; u < ROWS; ++u) {
                        const int k0 = pair_eval<FORM, UNIFORM>(R[u], a0, b0, n0, h0);
                        const int k1 = pair_eval<FORM, UNIFORM>(R[u], a1, b1, n1, h1);
                        R[u].m = __vimin3_s32(R[u].m, k0, k1);
                    }
                }
            };
            if (cnt == kColTile) {   // full stage: constant trip count
#pragma unroll 1
                for (int j0 = 0; j0 < kColTile; j0 += kColsPerIter) cols(j0);
            } else {
#pragma unroll 1
                for (int j0 = 0; j0 < cnt; j0 += kColsPerIter) cols(j0);     // cnt is a multiple of 8
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sh.empty_bar[s]);
        v += cnt;
    }
    kring = k;
#pragma unroll
    for (int u = 0; u < ROWS; ++u) {
        const int r = u * kBulkThreads + tid;
        int ov = veto_from_min<UNIFORM>(R[u].m, R[u].h, p.ov_tol);
        if (ov < 0)
            ov = r < nrows ? recheck_overlap_cg(p.xy, p.zq, p.hh, p.txy[row0 + r], p.tz[row0 + r], R[u].h, v0, v1, cbeg, gapv, gap) : 0;
        if (r < nrows) accum_row(p, row0 + r, R[u].acc, ov);
    }
}

}  // namespace mcb

namespace mcb {

// ------------------------------------------------------------------------------------------
// helper warp of the chain CTA: prepares row tile t of chunk c and hands it over
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void chain_helper_tile(const PArgs& a, PShared& sh, const ChunkBufs& B, int c, int t,
                                                  int row0, int gt, bool first) {
    const int lane = threadIdx.x & 31;
    const int C = a.C, W = C / kTile;
    const int r = t * kTile + lane, i = row0 + r;
    const int slot = gt % kRing;
    HandOff& ho = sh.u.ho[slot];
    const unsigned apar = (unsigned)(c >> 1) & 1u;
    const Watch wd{a.sy, a.p.st, a.p.wait_limit_ns};

    // what depends on the trial phase and the chunk's DIAG items only
    unsigned veto = (unsigned)a.p.wall[i];
    const double lbq = a.p.lbq[i], lnu = a.p.lnu[i];
    const double2 txy = a.p.txy[i];
    const double tz = a.p.tz[i];
    const unsigned ovoD = __ldcg(B.OVold + (size_t)r * W + t), ovnD = __ldcg(B.OVnew + (size_t)r * W + t);
    unsigned ovoP = 0u, ovnP = 0u;
    if (t > 0) { ovoP = __ldcg(B.OVold + (size_t)r * W + t - 1); ovnP = __ldcg(B.OVnew + (size_t)r * W + t - 1); }

    bool staged = false;
    auto stage_blocks = [&]() {
        // the slot is free once the publisher is done with tile gt - kRing.  A parity wait alone would be fooled if
        // this warp were two tiles of the slot ahead of the publisher (it can be, at the start of a chunk), so the
        // monotonic tile counter is checked first; the mbarrier then only orders the publisher's reads before the copy
        if (gt >= kRing) {
            if (*(volatile int*)&sh.pub_gt < gt - kRing + 1) {
                const unsigned long long t0 = global_ns();
                for (unsigned it = 1; *(volatile int*)&sh.pub_gt < gt - kRing + 1; ++it) {
                    __nanosleep(32);
                    if ((it & 1023u) == 0u) wd_check(wd, t0);
                }
            }
            mbar_wait_wd(wd, &sh.p_bar[slot], (unsigned)(gt / kRing - 1) & 1u);
        }
        if (lane == 0) {
            const int nb = min(t, 2) + 1;          // blocks (t, t-2), (t, t-1), (t, t): contiguous in Dblk
            const double* src = B.Dblk + (size_t)blk_index(t, t + 1 - nb) * (kTile * kTile);
            const uint32_t bytes = (uint32_t)nb * kTile * kTile * 8u;
            fence_proxy_async();
            mbar_arrive_expect_tx(&sh.d_bar[slot], bytes);
            bulk_g2s(ho.D + (3 - nb) * kTile * kTile, src, bytes, &sh.d_bar[slot]);
        }
        staged = true;
    };

#ifndef MCB_PRESTAGE
#define MCB_PRESTAGE 1
#endif
    if (first) {
        // this helper's first tile of the chunk: the block copy is under way while the chunk's last FAR and
        // urgent items complete (every lane polls -- one broadcast load: the warp waits, and gives up, as a whole)
        if (MCB_PRESTAGE) stage_blocks();
        const long long t0 = clock64();
        spin_until_ge(wd, sy_far_done(a) + c, far_items(a.p.Np, C, a.farcols, a.nfar, c));
        const long long t1 = clock64();
        if (c > 0) spin_until_ge(wd, sy_fix_done(a) + c, urgent_items(C, c, a.fixcols));
        if (t == 0 && lane == 0 && a.dbg) {
            a.dbg[3] += t1 - t0; a.dbg[4] += clock64() - t1;
            if (c < 300) a.dbg[16 + 3 * c] = (long long)global_ns();   // inputs of chunk c complete
        }
    }
    // base sum of all FAR, FIX and DIAG items of this row
    double E = accum_value(__ldcg(a.p.S1 + i), __ldcg(a.p.S2 + i));
    if (__ldcg(a.p.ovc + i) > 0) veto |= kFlagOverlap;

    // corrections of the column tiles s <= t - 3, as their accept masks appear (masked loads from L2)
    for (int s = 0; s + 3 <= t; ++s) {
        if (!staged && s + kRing >= t) stage_blocks();
        mbar_wait_wd(wd, &sh.a_bar[c & 1][s], apar);
        const unsigned A = sh.sA[c & 1][s];
        const double* blk = B.Dblk + (size_t)blk_index(t, s) * (kTile * kTile);
        double v[kTile];
#pragma unroll
        for (int jj = 0; jj < kTile; ++jj) v[jj] = ((A >> jj) & 1u) ? __ldcg(blk + jj * kTile + lane) : 0.0;
        const unsigned on = __ldcg(B.OVnew + (size_t)r * W + s), oo = __ldcg(B.OVold + (size_t)r * W + s);
        double s4[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int jj = 0; jj < kTile; ++jj) s4[jj & 3] = __dadd_rn(s4[jj & 3], v[jj]);
        E = __dadd_rn(E, __dadd_rn(__dadd_rn(s4[0], s4[1]), __dadd_rn(s4[2], s4[3])));
        if (((on & A) | (oo & ~A)) != 0u) veto |= kFlagOverlap;
    }
    if (!staged) stage_blocks();
    if (t >= 2) {
        // column tile t - 2, decided one tile ago: its block is already in the slot, so that only shared-memory
        // latency lies between the mask and the hand-over
        const int s = t - 2;
        const unsigned on = __ldcg(B.OVnew + (size_t)r * W + s), oo = __ldcg(B.OVold + (size_t)r * W + s);
        mbar_wait_wd(wd, &sh.d_bar[slot], (unsigned)(gt / kRing) & 1u);
        double v[kTile];
#pragma unroll
        for (int jj = 0; jj < kTile; ++jj) v[jj] = ho.D[jj * kTile + lane];
        mbar_wait_wd(wd, &sh.a_bar[c & 1][s], apar);
        const unsigned A = sh.sA[c & 1][s];
        double s8[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int jj = 0; jj < kTile; ++jj) s8[jj & 7] = __dadd_rn(s8[jj & 7], ((A >> jj) & 1u) ? v[jj] : 0.0);
        E = __dadd_rn(E, __dadd_rn(__dadd_rn(__dadd_rn(s8[0], s8[1]), __dadd_rn(s8[2], s8[3])),
                                  __dadd_rn(__dadd_rn(s8[4], s8[5]), __dadd_rn(s8[6], s8[7]))));
        if (((on & A) | (oo & ~A)) != 0u) veto |= kFlagOverlap;
    }

    ho.E[lane] = E; ho.lbq[lane] = lbq; ho.lnu[lane] = lnu;
    ho.txy[lane] = txy; ho.tz[lane] = tz;
    ho.ovoP[lane] = ovoP; ho.ovnP[lane] = ovnP; ho.ovoD[lane] = ovoD; ho.ovnD[lane] = ovnD;
    ho.veto[lane] = veto;
    __syncwarp();
    if (lane == 0) mbar_arrive(&sh.ho_bar[slot]);
}

// ------------------------------------------------------------------------------------------
// publisher warp of the chain CTA (a4): commit x <- x~ for the accepted trials, trial log, counters,
// and the progress counter the workers' FIX and release conditions read
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void chain_publisher(const PArgs& a, PShared& sh) {
    const int lane = threadIdx.x & 31;
    const Params& p = a.p;
    const int C = a.C, GPC = C / kGroup, ntfull = C / kTile;
    const Watch wd{a.sy, a.p.st, a.p.wait_limit_ns};
    unsigned long long n_acc = 0, n_ov = 0, n_wall = 0, n_tie = 0;
    double e_lane = 0.0;
    for (int c = 0; c < a.nchunks; ++c) {
        const int row0 = c * C, nt = chunk_rows(p.Np, C, c) / kTile;
        for (int t = 0; t < nt; ++t) {
            const int gt = c * ntfull + t, slot = gt % kRing;
            mbar_wait_wd(wd, &sh.a_bar[c & 1][t], (unsigned)(c >> 1) & 1u);
            const HandOff& ho = sh.u.ho[slot];
            const int i = row0 + t * kTile + lane;
            const unsigned fl = ho.out_flags[lane];
            const double dE = ho.out_dE[lane];
            const double2 t2 = ho.txy[lane];
            const double tz = ho.tz[lane];
            __syncwarp();
            if (lane == 0) {      // the slot is free for tile gt + kRing before the global stores below
                mbar_arrive(&sh.p_bar[slot]);
                *(volatile int*)&sh.pub_gt = gt + 1;
            }
            if (fl & kFlagAccept) {
                p.xy[i] = t2;
                p.zq[i].x = tz;
                p.nn[i] = dist2(t2.x, t2.y, tz);
                e_lane = __dadd_rn(e_lane, dE);
            }
            p.log_dE[i] = dE;
            p.log_flags[i] = (unsigned char)fl;
            if (i < p.N) {
                n_acc += (fl & kFlagAccept) ? 1 : 0;
                n_ov += (fl & kFlagOverlap) ? 1 : 0;
                n_wall += (fl & kFlagWall) ? 1 : 0;
                n_tie += (fl & kFlagNearTie) ? 1 : 0;
            }
            __syncwarp();
            if (lane == 0) {
                const int rows_done = (t + 1) * kTile;
                if (rows_done % kGroup == 0 || t + 1 == nt) {
                    __threadfence();
                    fence_proxy_async();
                    st_release(a.sy + kSyGroups, c * GPC + (rows_done + kGroup - 1) / kGroup);
                }
            }
        }
    }
    // fixed-order reductions over the lanes
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        n_acc += __shfl_xor_sync(0xffffffffu, n_acc, o);
        n_ov += __shfl_xor_sync(0xffffffffu, n_ov, o);
        n_wall += __shfl_xor_sync(0xffffffffu, n_wall, o);
        n_tie += __shfl_xor_sync(0xffffffffu, n_tie, o);
    }
    const double e_run = warp_sum(e_lane);
    if (lane == 0) {
        DevState* st = p.st;
        st->accepted += n_acc;
        st->veto_overlap += n_ov;
        st->veto_wall += n_wall;
        st->near_ties += n_tie;
        st->E_run += e_run;
        st->sweep += 1ull;
    }
}

}  // namespace mcb

namespace mcb {

// ------------------------------------------------------------------------------------------
// the chain CTA (a3/a4): Alg. 4; accept iff no veto and
// l_B q_i sum + ln u < 0 (Eq. 1 in log form, strict; readings G3, G4)
// ------------------------------------------------------------------------------------------
static __device__ __noinline__ void chain_cta(const PArgs& a, PShared& sh) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const Params& p = a.p;
    const int C = a.C;
    const int ntfull = C / kTile;
    const Watch wd{a.sy, a.p.st, a.p.wait_limit_ns};

    if (warp == kHelpers + 1) {
        chain_publisher(a, sh);
        return;
    }
    if (warp >= 1) {
        // ---------------- helpers ----------------
        const int h = warp - 1;
        for (int c = 0; c < a.nchunks; ++c) {
            const int row0 = c * C, nrows = chunk_rows(p.Np, C, c), nt = nrows / kTile;
            if (h >= nt) continue;
            {
                const long long t0 = clock64();
                spin_until_ge(wd, sy_diag_done(a) + c, diag_items(nrows, a.dsplit));
                if (h == 0 && lane == 0 && a.dbg) a.dbg[15] += clock64() - t0;
            }
            const ChunkBufs B = chunk_bufs(a, c);
            for (int t = h; t < nt; t += kHelpers) chain_helper_tile(a, sh, B, c, t, row0, c * ntfull + t, t == h);
        }
        return;
    }

    // ---------------- the chain warp ----------------
    if (a.mode == 2) return;   // watchdog test ("probe" = 2): nobody decides, the publisher's first wait runs into the limit
    long long w_first = 0, w_other = 0;
    const long long t_start = clock64();
    for (int c = 0; c < a.nchunks; ++c) {
        const int nt = chunk_rows(p.Np, C, c) / kTile;
        unsigned Ap = 0u;
        for (int t = 0; t < nt; ++t) {
            const int gt = c * ntfull + t, slot = gt % kRing;
            const long long tw = clock64();
            mbar_wait_wd(wd, &sh.ho_bar[slot], (unsigned)(gt / kRing) & 1u);
            if (t == 0) w_first += clock64() - tw; else w_other += clock64() - tw;
            if (t == 0 && lane == 0 && a.dbg && c < 300) a.dbg[16 + 3 * c + 1] = (long long)global_ns();   // chain starts chunk c
            mbar_wait_wd(wd, &sh.d_bar[slot], (unsigned)(gt / kRing) & 1u);   // (complete long ago; makes the copy visible here)
            HandOff& ho = sh.u.ho[slot];
            // the tile's two nearest blocks, one row each per lane, into registers: every pass below is then pure arithmetic
            double dp[kTile], dd[kTile];
            {
                const double* prev = ho.D + kTile * kTile;
                const double* diag = ho.D + 2 * kTile * kTile;
#pragma unroll
                for (int j = 0; j < kTile; ++j) { dp[j] = prev[j * kTile + lane]; dd[j] = diag[j * kTile + lane]; }   // dd: 0 for lanes <= j
            }
            const double lbq = ho.lbq[lane], lnu = ho.lnu[lane];
            double Eu = ho.E[lane];
            const unsigned vflags = ho.veto[lane];
            const bool wallv = (vflags & kFlagWall) != 0u;
            bool ovv = (vflags & kFlagOverlap) != 0u;
            auto masked_sum = [](const double (&d)[kTile], unsigned A) {
                double s8[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
                for (int j = 0; j < kTile; ++j) s8[j & 7] = __dadd_rn(s8[j & 7], ((A >> j) & 1u) ? d[j] : 0.0);
                return __dadd_rn(__dadd_rn(__dadd_rn(s8[0], s8[1]), __dadd_rn(s8[2], s8[3])),
                                 __dadd_rn(__dadd_rn(s8[4], s8[5]), __dadd_rn(s8[6], s8[7])));
            };
            if (t > 0) {  // corrections of the tile just resolved: block (t, t-1)
                Eu = __dadd_rn(Eu, masked_sum(dp, Ap));
                ovv = ovv || (((ho.ovnP[lane] & Ap) | (ho.ovoP[lane] & ~Ap)) != 0u);
            }
            // Decisions of the 32 trials of this tile.  Trial l depends on the accept bits of the lanes j < l only
            // (D(l, j) and the overlap bits are zero for j >= l), so the accept mask A is the unique fixed point of
            //   A = F(A),  F(A)_l = [ no veto given A  and  ln u_l + l_B q_l (E0_l + sum_j A_j D(l, j)) < 0 ]
            // and iterating F from any start fixes lane 0 in the first pass, lane 1 in the second, ...: at most 32
            // passes, in practice one or two (the corrections D are tiny against |dE + ln u| except near a tie),
            // each a masked sum instead of Alg. 4's 32 dependent steps.  Es < 0 is read off the
            // sign bit (Es is never -0: ln u < 0 strictly and an exact cancellation gives +0).
            const unsigned ovo = ho.ovoD[lane], ovn = ho.ovnD[lane];
            const double E0 = Eu;
            const bool veto0 = wallv || ovv;
            double Es = __fma_rn(lbq, E0, lnu);
            unsigned A = __ballot_sync(0xffffffffu, !veto0 && (__double2hiint(Es) < 0));
            bool hit = false;
#pragma unroll 1
            for (int pass = 0; pass <= kTile; ++pass) {
                Eu = __dadd_rn(E0, masked_sum(dd, A));
                Es = __fma_rn(lbq, Eu, lnu);
                hit = ((ovn & A) | (ovo & ~A)) != 0u;             // bits >= lane are 0 in both words
                const unsigned A1 = __ballot_sync(0xffffffffu, !veto0 && !hit && (__double2hiint(Es) < 0));
                if (A1 == A) break;
                A = A1;
            }
            const bool veto = veto0 || hit;
            ovv = ovv || hit;
            const bool acc = ((A >> lane) & 1u) != 0u;
            const bool tie = !veto && (fabs(Es) < 1e-8);
            ho.out_dE[lane] = __dmul_rn(lbq, Eu);
            ho.out_flags[lane] = (acc ? kFlagAccept : 0u) | (ovv ? kFlagOverlap : 0u) | (wallv ? kFlagWall : 0u) |
                                 (tie ? kFlagNearTie : 0u);
            Ap = A;
            if (lane == 0) sh.sA[c & 1][t] = A;
            __syncwarp();
            if (lane == 0) mbar_arrive(&sh.a_bar[c & 1][t]);
        }
        if (lane == 0 && a.dbg && c < 300) a.dbg[16 + 3 * c + 2] = (long long)global_ns();   // chain ends chunk c
    }
    if (lane == 0 && a.dbg) {
        a.dbg[0] = clock64() - t_start;   // chain warp: whole sweep
        a.dbg[1] = w_first;               //   waiting for the first tile of a chunk
        a.dbg[2] = w_other;               //   waiting for the other tiles (helpers late)
    }
}

}  // namespace mcb

namespace mcb {

enum { kItemExit = 0, kItemDiag = 1, kItemFarL = 2, kItemFix = 3, kItemFarU = 4, kItemMid = 5 };

// Work queues.  Each is a ticket counter in global memory; tickets run through the chunks in order.
//   QL  FAR-L items over the columns before chunk c-2 (final positions): released when the chain
//       has finished chunk c-3
//   QU  FAR-U items over the columns after chunk c (sweep-start positions): never blocked -- the
//       filler that keeps every SM busy while the chain works
//   QD  DIAG items: released when the chain has finished chunk c - kDRing (ring of D buffers)
//   FIX / MID urgent items: exist as soon as the chain has published their columns
// Thread 0 of a worker CTA reads all five words (four counters and the chain's progress) in one
// round trip, picks the first queue whose next ticket is released -- FIX/MID, QD, QL, QU for the
// FAR workers (what the chain needs soonest first); FIX/MID, QD for the a.nnear "near" workers that
// keep the latency of what the chain waits for short -- and claims with one atomic.  A ticket is claimed only when its chunk is released
// (a claim that races across a chunk boundary into an unreleased chunk is kept and run first once
// released), so no CTA sits on work that another CTA could do.
enum { QL = 0, QU = 1, QD = 2 };
struct Cursor {
    int c, base;    // chunk that holds the queue's next ticket, first ticket of that chunk
    int held;       // ticket claimed at a chunk boundary before its chunk was released (-1: none)
};
struct Cursors {
    Cursor l, u, d;
    int uunit;      // first urgent release unit this CTA has not seen exhausted
};

template <int Q>
__device__ __forceinline__ int items_of(const PArgs& a, int c) {
    return Q == QL ? far_slices(farL_cols(a.C, c), a.farcols, a.nfar)
         : Q == QU ? far_slices(a.mode == 1 ? probe_cols(a.p.Np, a.C, c) : farU_cols(a.p.Np, a.C, c), a.farcols, a.nfar)
                   : diag_items(chunk_rows(a.p.Np, a.C, c), a.dsplit);
}
template <int Q>
__device__ __forceinline__ void advance(const PArgs& a, Cursor& cur, int t) {
    while (cur.c < a.nchunks && t >= cur.base + items_of<Q>(a, cur.c)) {
        cur.base += items_of<Q>(a, cur.c);
        ++cur.c;
    }
}
// QL items of chunk c need the chain to have finished chunk c-3, QD items chunk c - kDRing (buffer ring)
template <int Q>
__device__ __forceinline__ bool released(const PArgs& a, int c, int groups) {
    return Q == QL ? (c < 3 || groups >= (c - 2) * (a.C / kGroup)) : (c < kDRing || groups >= (c - kDRing + 1) * (a.C / kGroup));
}

// t = the counter's value as just read, groups = the chain's progress as just read.
// true if an item of queue Q was claimed (written to item[]); done = queue exhausted
template <int Q>
__device__ __forceinline__ bool try_queue(const PArgs& a, Cursor& cur, int t, int groups, int* item, bool& done) {
    int* counter = a.sy + (Q == QL ? kSyTicket : Q == QU ? kSyTicketU : kSyDTicket);
    int mine = cur.held;
    if (mine < 0) {
        advance<Q>(a, cur, t);
        done = cur.c >= a.nchunks;
        if (done || (Q != QU && !released<Q>(a, cur.c, groups))) return false;
        mine = atomicAdd(counter, 1);
        advance<Q>(a, cur, mine);
        done = cur.c >= a.nchunks;
        if (done) return false;
    }
    done = false;
    if (Q != QU && !released<Q>(a, cur.c, groups)) {
        cur.held = mine;
        return false;
    }
    cur.held = -1;
    item[0] = Q == QL ? kItemFarL : Q == QU ? kItemFarU : kItemDiag;
    item[1] = cur.c;
    item[2] = mine - cur.base;
    return true;
}

__device__ __forceinline__ int ld_relaxed(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

static __device__ __noinline__ void fetch_item(const PArgs& a, Cursors& cur, bool near, int* item) {
    const int C = a.C, GPC = C / kGroup, nmid = C / kMidCols;
    const int total_units = urgent_units(C, a.nchunks), nper = kGroup / a.fixcols;
    int* sy = a.sy;
    for (unsigned it = 1;; ++it) {
        // no time limit of its own: leaves when another wait gave up -- through an exit ITEM, not by exiting: the
        // other threads of the CTA wait for the item at a barrier and would run the previous one again
        if ((it & 1023u) == 0u && *(volatile int*)(sy + kSyAbort) != 0) { item[0] = kItemExit; return; }
        // one round trip: five independent loads
        const int tl = ld_relaxed(sy + kSyTicket), tu = ld_relaxed(sy + kSyTicketU), td = ld_relaxed(sy + kSyDTicket);
        const int hint = ld_relaxed(sy + kSyUTicket), groups = ld_acquire(sy + kSyGroups);   // acquire: what the chain published
        bool got = false, l_done = true, u_done = true, d_done = false;
        if (a.mode == 1) {
            got = try_queue<QU>(a, cur.u, tu, groups, item, u_done);
            if (!got) item[0] = kItemExit;
            return;
        }
        // urgent items: walk the release units from the first one not known to be exhausted (this CTA's own
        // knowledge or the shared hint), stop at the first unit the chain has not released yet
        int k = max(cur.uunit, hint);
        while (k < total_units) {
            int c, g, mid;                         // unit k -> chunk c, MID unit or FIX group g
            if (k < GPC) { c = 1; g = k; mid = 0; }
            else { c = 2 + (k - GPC) / (GPC + 1); g = (k - GPC) % (GPC + 1) - 1; mid = g < 0 ? 1 : 0; }
            const int need = mid ? (c - 1) * GPC : (c - 1) * GPC + g + 1;
            if (groups < need) break;
            const int size = mid ? nmid : nper;
            const int v = atomicAdd(a.uc + k, 1);
            if (v < size) {
                item[0] = mid ? kItemMid : kItemFix; item[1] = c; item[2] = mid ? v : g * nper + v;
                got = true;
                if (v == size - 1) atomicMax(sy + kSyUTicket, k + 1);     // the hint for everybody else
                break;
            }
            ++k;
        }
        cur.uunit = k;
        if (!got) got = try_queue<QD>(a, cur.d, td, groups, item, d_done);
        if (!got && !near) got = try_queue<QL>(a, cur.l, tl, groups, item, l_done);
        if (!got && !near) got = try_queue<QU>(a, cur.u, tu, groups, item, u_done);
        if (got) return;
        if (l_done && u_done && d_done && k >= total_units) { item[0] = kItemExit; return; }
        __nanosleep(near ? 400 : 200);
    }
}

// DIAG item k of chunk c: 8 / dsplit units (row tile, column tile), each shared by dsplit warps that take
// 32 / dsplit of its columns each (small systems: more, shorter items -- the eta scheme of PAPER.md:243-245)
static __device__ __noinline__ void diag_item(const PArgs& a, PShared& sh, int c, int k, int row0, int nrows) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const ChunkBufs B = chunk_bufs(a, c);
    Params pc = a.p;
    pc.chunk = a.C;
    pc.Dblk = B.Dblk; pc.OVold = B.OVold; pc.OVnew = B.OVnew;
    const int split = a.dsplit, part = warp % split, per = kTile / split;
    const int unit = (k * 8 + warp) / split;
    unsigned ovo, ovn;
    diag_unit(pc, row0, nrows, unit, sh.u.w.cxy[warp], sh.u.w.czq[warp], sh.u.w.ctxy[warp], sh.u.w.ch[warp],
              sh.u.w.ctz[warp], part * per, (part + 1) * per, ovo, ovn);
    // the parts' overlap bits, combined by the first warp of the unit
    sh.u.w.ov[warp][0][lane] = ovo;
    sh.u.w.ov[warp][1][lane] = ovn;
    __syncthreads();
    const int nt = nrows / kTile;
    if (part == 0 && unit < nt * nt) {
        for (int q = 1; q < split; ++q) { ovo |= sh.u.w.ov[warp + q][0][lane]; ovn |= sh.u.w.ov[warp + q][1][lane]; }
        const int t = unit / nt, s2 = unit % nt;
        if (s2 <= t) {
            const int W = a.C / kTile, r = t * kTile + lane;
            B.OVold[(size_t)r * W + s2] = ovo;
            B.OVnew[(size_t)r * W + s2] = ovn;
        }
    }
}

// Grid-wide barrier between the phases of a launch (all CTAs are co-resident: cooperative launch).  Arrivals are
// counted in gbar[0]; the last one resets the count and releases the others by bumping the generation gbar[32].
// The acquire load (LDG.STRONG.GPU + CCTL.IVALL) also drops this SM's L1, so plain loads after the barrier see
// what the other CTAs wrote before it.
__device__ __forceinline__ bool grid_barrier(const PArgs& a, PShared& sh) {
    __syncthreads();
    if (threadIdx.x == 0) {
        const Watch wd{a.sy, a.p.st, a.p.wait_limit_ns};
        int* cnt = a.gbar;
        int* gen = a.gbar + 32;
        int ok = 1;
        const int g0 = ld_acquire(gen);          // read before arriving: nobody can bump it until this CTA has arrived
        __threadfence();
        if (atomicAdd(cnt, 1) == (int)gridDim.x - 1) {
            *(volatile int*)cnt = 0;
            __threadfence();
            st_release(gen, g0 + 1);
        } else {
            const unsigned long long t0 = global_ns();
            for (unsigned it = 1; ld_acquire(gen) == g0; ++it) {
                __nanosleep(40);
                if ((it & 1023u) == 0u && wd_poll(wd, t0)) { ok = 0; break; }
            }
        }
        sh.item[3] = (sh.item[3] & 1) | (ok ? 0 : 2);   // bit 1: the launch is being abandoned (a wait ran into the watchdog)
    }
    __syncthreads();
    return (sh.item[3] & 2) == 0;      // the same in every thread of the CTA: they leave the kernel together
}

// a1 for the whole system, shared out over all threads of the grid; also clears the row accumulators
static __device__ __noinline__ void trial_phase(const Params& p) {
    const unsigned long long s = *(volatile unsigned long long*)&p.st->sweep;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < p.Np; i += gridDim.x * blockDim.x) trial_one(p, i, s);
}

// the worker loop of one sweep: pull items until every queue is exhausted
template <int ROWS, bool UNIFORM, int FORM>
__device__ __forceinline__ void worker_sweep(const PArgs& a, PShared& sh, unsigned& kring) {
    const int tid = threadIdx.x, warp = tid >> 5;
    const Params& p = a.p;
    const int C = a.C;
    Cursors cur{{0, 0, -1}, {0, 0, -1}, {0, 0, -1}, 0};
    if (a.dbg && blockIdx.x == 1 && tid == 0) a.dbg[16 + 3 * 300 + 40] = (long long)global_ns();
    const bool near = (int)blockIdx.x <= a.nnear;
    for (;;) {
        __syncthreads();
        if (tid == 0) {
            const long long t0 = clock64();
            fetch_item(a, cur, near, sh.item);
            if (a.dbg) {
                atomicAdd((unsigned long long*)a.dbg + 5, (unsigned long long)(clock64() - t0));
                if (!near) {   // FAR workers' fetch time by 0.5 ms bucket since the first chunk's start
                    const long long origin = *(volatile long long*)(a.dbg + 16 + 3 * 300 + 40);
                    const int bkt = origin ? (int)min(31ull, (global_ns() - (unsigned long long)origin) / 500000ull) : 0;
                    atomicAdd((unsigned long long*)a.dbg + 16 + 3 * 300 + bkt, (unsigned long long)(clock64() - t0));
                }
                atomicAdd((unsigned long long*)a.dbg + 6 + (sh.item[0] == kItemMid ? kItemFix : sh.item[0]), 1ull);   // [6] exits, [7] diag, [8] farL, [9] fix, [10] farU
            }
        }
        __syncthreads();
        const int type = sh.item[0], c = sh.item[1], k = sh.item[2];
        const long long t_item = clock64();
        if (type == kItemExit) break;
        const int row0 = c * C, nrows = chunk_rows(p.Np, C, c);
        if (type == kItemDiag) {
            if (warp < 8) diag_item(a, sh, c, k, row0, nrows);
        } else {
            // one call site for the pair loop: the item's column space [cb, cb + ...) minus [g0, g1), columns [v0, v1) of it
            int cb, g0, g1, v0, v1;
            if (type == kItemFarL || type == kItemFarU) {
                // before chunk c-2 (L) or after chunk c (U); probe: all columns but the chunk's own
                const bool probe = a.mode == 1;
                cb = (type == kItemFarL || probe) ? 0 : row0 + nrows;
                const int ncols = probe ? probe_cols(p.Np, C, c) : type == kItemFarL ? farL_cols(C, c) : farU_cols(p.Np, C, c);
                const int nf = far_slices(ncols, a.farcols, a.nfar);
                v0 = slice_bound(ncols, nf, k); v1 = slice_bound(ncols, nf, k + 1);
                g0 = probe ? row0 : cb; g1 = probe ? row0 + nrows : cb;
            } else {
                const int w = type == kItemMid ? kMidCols : a.fixcols;
                cb = row0 - (type == kItemMid ? 2 : 1) * C + k * w;
                g0 = g1 = cb; v0 = 0; v1 = w;
            }
            bulk_item<ROWS, UNIFORM, FORM>(p, sh, kring, row0, nrows, cb, g0, g1, v0, v1);
        }
        __syncthreads();
        if (tid == 0) {
            // completion counter of this item's queue and chunk (item[] is stable until the next fetch)
            const int ty = ((volatile int*)sh.item)[0], cc = ((volatile int*)sh.item)[1];
            int* done = (ty == kItemDiag ? sy_diag_done(a) : (ty == kItemFix || ty == kItemMid) ? sy_fix_done(a) : sy_far_done(a)) + cc;
            __threadfence();
            atomicAdd(done, 1);
            if (a.dbg) {
                const unsigned long long dt = (unsigned long long)(clock64() - t_item);
                atomicAdd((unsigned long long*)a.dbg + 10 + (ty == kItemFarU ? kItemFarL : ty == kItemMid ? kItemFix : ty), dt);   // busy cycles: [11] diag [12] far [13] fix
                if (near) atomicAdd((unsigned long long*)a.dbg + 14, dt);                              // [14] near workers
            }
        }
    }
}

// One launch = a.nsweeps full sweeps.  Per sweep: trial generation by the whole grid (a1), grid barrier, the sweep
// proper (chain CTA + workers, a2-a4), grid barrier, reset of the scheduling words.  mc_sweep(n) is therefore one
// launch whatever n is (PAPER.md:85-91 launched one kernel per cycle and generated the random numbers on the host).
template <int ROWS, bool UNIFORM, int FORM>
__global__ void __launch_bounds__(kPThreads, 2) k_sweep(const PArgs a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    PShared& sh = *reinterpret_cast<PShared*>(smem_raw);
    const int tid = threadIdx.x;
    const Params& p = a.p;
    if (*(volatile int*)&p.st->stall) return;   // a stalled sweep invalidated the state: every later sweep is a no-op

    auto init_chain_barriers = [&]() {
        for (int s = 0; s < kRing; ++s) { mbar_init(&sh.ho_bar[s], 1); mbar_init(&sh.d_bar[s], 1); mbar_init(&sh.p_bar[s], 1); }
        for (int s = 0; s < 2 * (kChunkMax / kTile); ++s) mbar_init(&sh.a_bar[0][0] + s, 1);
        *(volatile int*)&sh.pub_gt = 0;
    };
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&sh.full_bar[s], 1);
            mbar_init(&sh.empty_bar[s], kPThreads / 32);
        }
        init_chain_barriers();
        mbar_fence_init();
        // the chain CTA gets its SM to itself: it publishes the SM it runs on, and the worker CTA
        // that shares that SM does no work in this launch (it only takes part in the grid barriers)
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        if (blockIdx.x == 0) {
            sh.item[3] = 0;
            st_release(a.sy + kSyChainSm, (int)smid + 1);
        } else {
            int v;
            const Watch wd{a.sy, a.p.st, a.p.wait_limit_ns};
            const unsigned long long t0 = global_ns();
            for (unsigned it = 1; (v = ld_acquire(a.sy + kSyChainSm)) == 0; ++it) {
                __nanosleep(100);
                if ((it & 1023u) == 0u) wd_check(wd, t0);
            }
            sh.item[3] = (v == (int)smid + 1) ? 1 : 0;
        }
    }
    __syncthreads();
    const bool is_chain = blockIdx.x == 0 && a.mode != 1;
    const bool idle = blockIdx.x != 0 && (sh.item[3] & 1) == 1 && a.mode != 1;

    unsigned kring = 0;
    for (int sw = 0; sw < a.nsweeps; ++sw) {
        trial_phase(p);
        if (!grid_barrier(a, sh)) return;
        if (is_chain) {
            if (sw > 0) {      // the hand-off barriers start every sweep in phase 0
                if (tid == 0) {
                    for (int s = 0; s < 3 * kRing + 2 * (kChunkMax / kTile); ++s)
                        asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&sh.ho_bar[0] + s)) : "memory");
                    init_chain_barriers();
                    mbar_fence_init();
                }
                __syncthreads();
            }
            chain_cta(a, sh);
        } else if (!idle) {
            worker_sweep<ROWS, UNIFORM, FORM>(a, sh, kring);
        }
        if (!grid_barrier(a, sh)) return;
        // everybody is done with the scheduling words: CTA 0 clears them for the next sweep (or the next launch);
        // the election word stays until the launch ends.  The next reader is behind the next grid barrier.
        if (blockIdx.x == 0) {
            // the protocol's own invariant: every item of the plan ran
            // exactly once -- each chunk's completion counters equal the item counts the plan gives for it
            if (a.mode == 0) {
                int bad = 0;
                for (int c = tid; c < a.nchunks; c += kPThreads) {
                    bad |= a.sy[kSyHdr + c] != far_items(p.Np, a.C, a.farcols, a.nfar, c);
                    bad |= a.sy[kSyHdr + a.nchunks + c] != diag_items(chunk_rows(p.Np, a.C, c), a.dsplit);
                    bad |= a.sy[kSyHdr + 2 * a.nchunks + c] != urgent_items(a.C, c, a.fixcols);
                }
                if (__syncthreads_or(bad) && tid == 0) p.st->sched_mismatch += 1;
            }
            // snapshot for mc_debug_peek, then clear
            const bool last = sw + 1 == a.nsweeps;
            for (int j = tid; j < p.sy_n; j += kPThreads) {
                a.sy[p.sy_n + j] = a.sy[j];
                if (last || j != kSyChainSm) a.sy[j] = 0;
            }
            for (int j = tid; j < urgent_units(a.C, a.nchunks); j += kPThreads) a.uc[j] = 0;
        }
    }
}

}  // namespace mcb
