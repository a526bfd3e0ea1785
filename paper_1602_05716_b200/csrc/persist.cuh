// persist.cuh -- one persistent kernel per sweep (sm_100a).  See DESIGN.md section 6.
//
// grid = 2 CTAs per SM, all co-resident (cooperative launch).  CTA 0 is the chain: it resolves the
// sweep's N decisions in ascending order.  Every other CTA is a worker that
// pulls items from two queues kept in global memory:
//   normal queue, in chunk order c = 0, 1, ...:
//     DIAG(c)  speculative corrections inside chunk c (as k_diag)                     (a2/a3)
//     FAR(c)   rows of chunk c x a slice of the columns outside chunks c-1 and c       (a2)
//              needs the chain to have finished chunk c-2
//   urgent queue:
//     FIX(c)   rows of chunk c x 16 columns of chunk c-1 at their final positions      (a2)
//              available as soon as the chain has published those columns' row group
// Partial sums go to fixed slots, so the result does not depend on which CTA ran which item.
// The chain CTA: warp 0 decides (ballot per step, as k_chain); warps 1..8 each own row tiles
// t = w-1 (mod 8): they gather the tile's base sum, add the corrections of all column tiles
// s <= t-2 as their accept masks appear, and hand the tile over through shared memory together
// with the two blocks D(t,t-1), D(t,t) the chain warp applies itself (one bulk copy).
#pragma once
#include "kernels.cuh"

namespace mcb {

constexpr int kPThreads = kBulkThreads + 32;   // 8 consumer warps + 1 producer warp
constexpr int kGroup = 128;                    // rows per published progress step of the chain
constexpr int kFixCols = 16;                   // columns per FIX item
constexpr int kRing = 4;                       // hand-off ring depth of the chain CTA
constexpr int kHelpers = 8;
constexpr int kMaxFixSlots = kChunkMax / kFixCols;

// scheduling state in global memory; zeroed by k_trial at the start of every sweep
enum { kSyTicket = 0, kSyUTicket = 1, kSyGroups = 2, kSyHdr = 4 };

struct PArgs {
    Params p;
    int C;            // rows per chunk = 256 * ROWS
    int nchunks;
    int nworkers;     // target number of FAR slices per chunk
    int* sy;          // [kSyHdr + 4 * nchunks]: header, far_done, far_ready, diag_done, fix_done
    double* Efar; int* ovfar;   // [2][kChunkMax]     reduced FAR sums of a chunk
    double* partF; int* ovF;    // [2][kMaxFixSlots][kChunkMax]
};

__host__ __device__ inline int chunk_rows(int Np, int C, int c) { return min(C, Np - c * C); }
__host__ __device__ inline int far_cols(int Np, int C, int c) {
    const int row0 = c * C, prev0 = c > 0 ? row0 - C : row0;
    return Np - (row0 + chunk_rows(Np, C, c) - prev0);
}
__host__ __device__ inline int far_slices(int ncols, int nworkers) {
    int n = ncols / 64;                      // at least 64 columns per slice
    if (n > nworkers) n = nworkers;
    if (n > kMaxSlices) n = kMaxSlices;
    if (n < 1 && ncols > 0) n = 1;
    return n;
}
__host__ __device__ inline int diag_items(int nrows) {
    const int nt = nrows / kTile;
    return (nt * nt + 7) / 8;
}
__host__ __device__ inline int normal_items(int Np, int C, int nworkers, int c) {
    return diag_items(chunk_rows(Np, C, c)) + far_slices(far_cols(Np, C, c), nworkers);
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

// shared memory of one CTA: workers use the column ring, the chain CTA the hand-off ring
struct HandOff {
    double D[2 * kTile * kTile];   // blocks (t, t-1) and (t, t), [jj][lane] each
    double E[kTile], lbq[kTile], lnu[kTile];
    double2 txy[kTile];
    double tz[kTile];
    unsigned ovoP[kTile], ovnP[kTile], ovoD[kTile], ovnD[kTile];
    unsigned veto[kTile];
};

struct __align__(128) PShared {
    union {
        struct {
            ColStage stage[kStages];
            double2 cxy[8][32], czq[8][32], ctxy[8][32];
            double ch[8][32], ctz[8][32];
        } w;
        HandOff ho[kRing];
    } u;
    uint64_t full_bar[kStages], empty_bar[kStages];
    uint64_t ho_bar[kRing];            // tile handed over (helper arrivals + bulk-copy bytes)
    uint64_t a_bar[2][kChunkMax / kTile]; // accept mask of tile t of a chunk (by chunk parity) published
    unsigned sA[2][kChunkMax / kTile];
    int item[4];
};

}  // namespace mcb

namespace mcb {

__device__ __forceinline__ double2 ldcg2(const double2* p) {
    double2 v;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}

// exact overlap re-check with L2 loads (columns may have been rewritten by the chain during this kernel)
__device__ __noinline__ int recheck_overlap_cg(const double2* xy, const double2* zq, const double* hh, double2 t,
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

// FAR / FIX item: all rows of the chunk (ROWS per consumer thread) x virtual columns [v0, v1) of
// [cbeg, cend) minus [gap0, gap1).  Same inner loop as k_bulk; the mbarrier ring persists across
// items (kring = stages used so far, identical in the producer and in every consumer).
template <int ROWS, bool UNIFORM>
__device__ __forceinline__ void bulk_item(const Params& p, PShared& sh, unsigned& kring, int row0, int nrows,
                                          int cbeg, int cend, int gap0, int gap1, int v0, int v1, double* part,
                                          int* ovout) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int kConsumerWarps = kBulkThreads / 32;
    const int gap = gap1 - gap0;
    const int gapv = gap0 - cbeg;
    (void)cend;

    if (warp == kConsumerWarps) {
        if (lane == 0) {
            fence_proxy_async();
            unsigned k = kring;
            for (int v = v0; v < v1; ++k) {
                const int lim = (v < gapv) ? min(v1, gapv) : v1;
                const int cnt = min(kColTile, lim - v);
                const int a = cbeg + ((v < gapv) ? v : v + gap);
                const unsigned s = k % kStages;
                if (k >= (unsigned)kStages) mbar_wait(&sh.empty_bar[s], ((k / kStages) - 1) & 1);
                mbar_arrive_expect_tx(&sh.full_bar[s], (uint32_t)cnt * (UNIFORM ? 32u : 40u));
                bulk_g2s(sh.u.w.stage[s].xy, p.xy + a, (uint32_t)cnt * 16u, &sh.full_bar[s]);
                bulk_g2s(sh.u.w.stage[s].zq, p.zq + a, (uint32_t)cnt * 16u, &sh.full_bar[s]);
                if (!UNIFORM) bulk_g2s(sh.u.w.stage[s].h, p.hh + a, (uint32_t)cnt * 8u, &sh.full_bar[s]);
                v += cnt;
            }
        }
        // every thread advances the ring counter identically
        for (int v = v0; v < v1; ++kring) {
            const int lim = (v < gapv) ? min(v1, gapv) : v1;
            v += min(kColTile, lim - v);
        }
        return;
    }

    RowRegs R[ROWS];
#pragma unroll
    for (int u = 0; u < ROWS; ++u) {
        const int r = u * kBulkThreads + tid;
        const int i = row0 + (r < nrows ? r : 0);
        const double2 xyi = ldcg2(p.xy + i);
        const double2 txyi = p.txy[i];
        R[u].x = xyi.x; R[u].y = xyi.y; R[u].z = __ldcg(&p.zq[i].x);
        const double Dx = __dadd_rn(txyi.x, -xyi.x), Dy = __dadd_rn(txyi.y, -xyi.y), Dz = __dadd_rn(p.tz[i], -R[u].z);
        R[u].ex = __dadd_rn(Dx, Dx); R[u].ey = __dadd_rn(Dy, Dy); R[u].ez = __dadd_rn(Dz, Dz);
        R[u].c = dist2(Dx, Dy, Dz);
        R[u].h = p.hh[i];
        R[u].acc = 0.0;
        R[u].m = 0x7fffffff;
    }
    const bool warp_live = warp * 32 < nrows;

    unsigned k = kring;
    for (int v = v0; v < v1; ++k) {
        const int lim = (v < gapv) ? min(v1, gapv) : v1;
        const int cnt = min(kColTile, lim - v);
        const unsigned s = k % kStages;
        mbar_wait(&sh.full_bar[s], (k / kStages) & 1);
        const ColStage& st = sh.u.w.stage[s];
        if (warp_live) {
#pragma unroll 1
            for (int j0 = 0; j0 < cnt; j0 += 4) {     // cnt is a multiple of 8
#pragma unroll
                for (int jj = 0; jj < 4; jj += 2) {
                    const double2 a0 = st.xy[j0 + jj], a1 = st.xy[j0 + jj + 1];
                    const double2 b0 = st.zq[j0 + jj], b1 = st.zq[j0 + jj + 1];
                    const double h0 = UNIFORM ? 0.0 : st.h[j0 + jj], h1 = UNIFORM ? 0.0 : st.h[j0 + jj + 1];
#pragma unroll
                    for (int u = 0; u < ROWS; ++u) {
                        const int k0 = pair_eval<UNIFORM>(R[u], a0, b0, h0);
                        const int k1 = pair_eval<UNIFORM>(R[u], a1, b1, h1);
                        R[u].m = __vimin3_s32(R[u].m, k0, k1);
                    }
                }
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
        int key = R[u].m;
        if (UNIFORM) {
            const double s = __dadd_rn(R[u].h, R[u].h);
            key -= __double2hiint(__dmul_rn(s, s));
        }
        int ov = key < 0 ? 1 : 0;
        if (r < nrows && key >= -kOvBand && key <= kOvBand)
            ov = recheck_overlap_cg(p.xy, p.zq, p.hh, p.txy[row0 + r], p.tz[row0 + r], R[u].h, v0, v1, cbeg, gapv, gap);
        if (r < nrows) {
            part[r] = R[u].acc;
            ovout[r] = ov;
        }
    }
}

}  // namespace mcb

namespace mcb {

// per-chunk view of the double-buffered scratch (parity b = c & 1)
struct ChunkBufs {
    double* partA; int* ovA;       // [slices][C]
    double* Efar; int* ovfar;      // [C]
    double* partF; int* ovF;       // [C / kFixCols][C]
    double* partD; int* ovD;       // [C / 32][C]
    double* Dblk;                  // [nt (nt + 1) / 2][32][32]
    unsigned* OVold; unsigned* OVnew;   // [C][C / 32]
};

__device__ __forceinline__ ChunkBufs chunk_bufs(const PArgs& a, int c) {
    const size_t b = (size_t)(c & 1);
    const size_t nt = kChunkMax / kTile;
    ChunkBufs B;
    B.partA = a.p.partA + b * kMaxSlices * kChunkMax;  B.ovA = a.p.ovA + b * kMaxSlices * kChunkMax;
    B.Efar = a.Efar + b * kChunkMax;                   B.ovfar = a.ovfar + b * kChunkMax;
    B.partF = a.partF + b * kMaxFixSlots * kChunkMax;  B.ovF = a.ovF + b * kMaxFixSlots * kChunkMax;
    B.partD = a.p.partD + b * nt * kChunkMax;          B.ovD = a.p.ovD + b * nt * kChunkMax;
    B.Dblk = a.p.Dblk + b * (nt * (nt + 1) / 2) * (kTile * kTile);
    B.OVold = a.p.OVold + b * kChunkMax * nt;          B.OVnew = a.p.OVnew + b * kChunkMax * nt;
    return B;
}

__device__ __forceinline__ int* sy_far_done(const PArgs& a) { return a.sy + kSyHdr; }
__device__ __forceinline__ int* sy_far_ready(const PArgs& a) { return a.sy + kSyHdr + a.nchunks; }
__device__ __forceinline__ int* sy_diag_done(const PArgs& a) { return a.sy + kSyHdr + 2 * a.nchunks; }
__device__ __forceinline__ int* sy_fix_done(const PArgs& a) { return a.sy + kSyHdr + 3 * a.nchunks; }

__device__ __forceinline__ void spin_until_ge(const int* p, int v) {
    while (ld_acquire(p) < v) __nanosleep(64);
}

// ------------------------------------------------------------------------------------------
// helper warp of the chain CTA: prepares row tile t of chunk c and hands it over
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void chain_helper_tile(const PArgs& a, PShared& sh, const ChunkBufs& B, int c, int t,
                                                  int row0, int nt, int nf, int nfix, int gt) {
    const int lane = threadIdx.x & 31;
    const int C = a.C, W = C / kTile;
    const int r = t * kTile + lane, i = row0 + r;
    const int slot = gt % kRing;
    HandOff& ho = sh.u.ho[slot];
    const unsigned apar = (unsigned)(c >> 1) & 1u;

    // base sum: FAR (reduced) + FIX slots + DIAG slots, fixed order
    double e4[4] = {0.0, 0.0, 0.0, 0.0};
    int ovc = 0;
    if (nf > 0) { e4[0] = __ldcg(B.Efar + r); ovc = __ldcg(B.ovfar + r); }
    for (int j = 0; j < nfix; j += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            e4[u] = __dadd_rn(e4[u], __ldcg(B.partF + (size_t)(j + u) * C + r));
            ovc += __ldcg(B.ovF + (size_t)(j + u) * C + r);
        }
    }
    for (int s = 0; s < nt; ++s) {
        e4[s & 3] = __dadd_rn(e4[s & 3], __ldcg(B.partD + (size_t)s * C + r));
        ovc += __ldcg(B.ovD + (size_t)s * C + r);
    }
    double E = __dadd_rn(__dadd_rn(e4[0], e4[1]), __dadd_rn(e4[2], e4[3]));
    unsigned veto = (unsigned)a.p.wall[i] | (ovc > 0 ? kFlagOverlap : 0u);

    // per-row scalars and the overlap words of the two blocks the chain warp applies itself
    const double lbq = a.p.lbq[i], lnu = a.p.lnu[i];
    const double2 txy = a.p.txy[i];
    const double tz = a.p.tz[i];
    const unsigned ovoD = __ldcg(B.OVold + (size_t)r * W + t), ovnD = __ldcg(B.OVnew + (size_t)r * W + t);
    unsigned ovoP = 0u, ovnP = 0u;
    if (t > 0) { ovoP = __ldcg(B.OVold + (size_t)r * W + t - 1); ovnP = __ldcg(B.OVnew + (size_t)r * W + t - 1); }

    bool staged = false;
    auto stage_blocks = [&]() {
        // the slot is free once the chain has finished tile gt - kRing
        if (gt >= kRing) {
            if (t >= kRing) mbar_wait(&sh.a_bar[c & 1][t - kRing], apar);
            else mbar_wait(&sh.a_bar[(c - 1) & 1][C / kTile + t - kRing], (unsigned)((c - 1) >> 1) & 1u);
        }
        if (lane == 0) {
            const double* src = B.Dblk + (size_t)blk_index(t, t > 0 ? t - 1 : 0) * (kTile * kTile);
            const uint32_t bytes = (t > 0 ? 2u : 1u) * kTile * kTile * 8u;
            fence_proxy_async();
            mbar_arrive_expect_tx(&sh.ho_bar[slot], bytes);
            bulk_g2s(t > 0 ? ho.D : ho.D + kTile * kTile, src, bytes, &sh.ho_bar[slot]);
        }
        staged = true;
    };

    // corrections of the column tiles s <= t - 2, as their accept masks appear
    for (int s = 0; s + 2 <= t; ++s) {
        if (!staged && s + kRing >= t) stage_blocks();   // a_bar[t - kRing] is awaited here at the latest
        mbar_wait(&sh.a_bar[c & 1][s], apar);
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

    ho.E[lane] = E; ho.lbq[lane] = lbq; ho.lnu[lane] = lnu;
    ho.txy[lane] = txy; ho.tz[lane] = tz;
    ho.ovoP[lane] = ovoP; ho.ovnP[lane] = ovnP; ho.ovoD[lane] = ovoD; ho.ovnD[lane] = ovnD;
    ho.veto[lane] = veto;
    __syncwarp();
    if (lane == 0) mbar_arrive(&sh.ho_bar[slot]);
}

}  // namespace mcb

namespace mcb {

// ------------------------------------------------------------------------------------------
// the chain CTA (a3/a4): Alg. 4; accept iff no veto and
// l_B q_i sum + ln u < 0 (Eq. 1 in log form, strict; readings G3, G4)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void chain_cta(const PArgs& a, PShared& sh) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const Params& p = a.p;
    const int C = a.C, GPC = C / kGroup;
    const int ntfull = C / kTile;

    if (warp >= 1) {
        // ---------------- helpers ----------------
        const int h = warp - 1;
        for (int c = 0; c < a.nchunks; ++c) {
            const int row0 = c * C, nrows = chunk_rows(p.Np, C, c), nt = nrows / kTile;
            const int nf = far_slices(far_cols(p.Np, C, c), a.nworkers);
            const int nfix = c > 0 ? C / kFixCols : 0;
            if (h >= nt) continue;
            if (lane == 0) {
                if (nf > 0) spin_until_ge(sy_far_ready(a) + c, 1);
                spin_until_ge(sy_diag_done(a) + c, diag_items(nrows));
                if (nfix > 0) spin_until_ge(sy_fix_done(a) + c, nfix);
            }
            __syncwarp();
            const ChunkBufs B = chunk_bufs(a, c);
            for (int t = h; t < nt; t += kHelpers) chain_helper_tile(a, sh, B, c, t, row0, nt, nf, nfix, c * ntfull + t);
        }
        return;
    }

    // ---------------- the chain warp ----------------
    unsigned long long n_acc = 0, n_ov = 0, n_wall = 0, n_tie = 0;
    double e_run = 0.0;
    for (int c = 0; c < a.nchunks; ++c) {
        const int row0 = c * C, nrows = chunk_rows(p.Np, C, c), nt = nrows / kTile;
        unsigned Ap = 0u;
        for (int t = 0; t < nt; ++t) {
            const int gt = c * ntfull + t, slot = gt % kRing;
            mbar_wait(&sh.ho_bar[slot], (unsigned)(gt / kRing) & 1u);
            const HandOff& ho = sh.u.ho[slot];
            const int i = row0 + t * kTile + lane;
            const double lbq = ho.lbq[lane], lnu = ho.lnu[lane];
            double Eu = ho.E[lane];
            const unsigned vflags = ho.veto[lane];
            const bool wallv = (vflags & kFlagWall) != 0u;
            bool ovv = (vflags & kFlagOverlap) != 0u;
            if (t > 0) {  // corrections of the tile just resolved: block (t, t-1)
                double s4[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
                for (int jj = 0; jj < kTile; ++jj)
                    if ((Ap >> jj) & 1u) s4[jj & 3] = __dadd_rn(s4[jj & 3], ho.D[jj * kTile + lane]);
                Eu = __dadd_rn(Eu, __dadd_rn(__dadd_rn(s4[0], s4[1]), __dadd_rn(s4[2], s4[3])));
                ovv = ovv || (((ho.ovnP[lane] & Ap) | (ho.ovoP[lane] & ~Ap)) != 0u);
            }
            double Es = __fma_rn(lbq, Eu, lnu);
            const unsigned ovo = ho.ovoD[lane], ovn = ho.ovnD[lane];
            const double* diag = ho.D + kTile * kTile;
            unsigned A = 0u;
#pragma unroll
            for (int j = 0; j < kTile; ++j) {
                const double dj = diag[j * kTile + lane];   // 0 for lanes <= j
                const double djs = __dmul_rn(lbq, dj);
                const bool ok = !wallv && !ovv && (Es < 0.0);
                const unsigned bal = __ballot_sync(0xffffffffu, ok);
                const bool bit = ((bal >> j) & 1u) != 0u;
                A |= (bit ? 1u : 0u) << j;
                if (bit) {
                    Es = __dadd_rn(Es, djs);
                    Eu = __dadd_rn(Eu, dj);
                }
                ovv = ovv || ((((bit ? ovn : ovo) >> j) & 1u) != 0u);  // bits >= lane are 0
            }
            const bool acc = ((A >> lane) & 1u) != 0u;
            const double dE = __dmul_rn(lbq, Eu);
            const bool tie = !wallv && !ovv && (fabs(Es) < 1e-8);
            if (acc) {   // commit: x <- x~ (a4)
                p.xy[i] = ho.txy[lane];
                p.zq[i].x = ho.tz[lane];
            }
            p.log_dE[i] = dE;
            p.log_flags[i] = (unsigned char)((acc ? kFlagAccept : 0u) | (ovv ? kFlagOverlap : 0u) |
                                             (wallv ? kFlagWall : 0u) | (tie ? kFlagNearTie : 0u));
            const bool real = i < p.N;
            n_acc += __popc(A);
            n_ov += __popc(__ballot_sync(0xffffffffu, real && ovv));
            n_wall += __popc(__ballot_sync(0xffffffffu, real && wallv));
            n_tie += __popc(__ballot_sync(0xffffffffu, real && tie));
            e_run += warp_sum(acc ? dE : 0.0);
            Ap = A;
            if (lane == 0) sh.sA[c & 1][t] = A;
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&sh.a_bar[c & 1][t]);
                // publish the committed rows to the workers, one group (or the chunk's end) at a time
                const int rows_done = (t + 1) * kTile;
                if (rows_done % kGroup == 0 || t + 1 == nt) {
                    __threadfence();
                    fence_proxy_async();
                    st_release(a.sy + kSyGroups, c * GPC + (rows_done + kGroup - 1) / kGroup);
                }
            }
        }
    }
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

enum { kItemExit = 0, kItemDiag = 1, kItemFar = 2, kItemFix = 3 };

// Thread 0 of a worker CTA: claim the next item.  Urgent items first; a claimed normal ticket whose
// chunk is not yet released by the chain is kept while urgent items are served (the chain can only
// be waiting for items that are already claimed or urgent, so nobody starves).
struct Cursor {
    int ticket;     // claimed normal ticket, -1 if none
    int c, base;    // chunk the ticket cursor is in, first ticket of that chunk
};

__device__ __forceinline__ void fetch_item(const PArgs& a, Cursor& cur, int* item) {
    const int C = a.C, GPC = C / kGroup, fix_per_chunk = C / kFixCols;
    const int total_urgent = (a.nchunks - 1) * fix_per_chunk;
    int* sy = a.sy;
    for (;;) {
        const int u = *(volatile int*)(sy + kSyUTicket);
        if (u < total_urgent) {
            const int c = 1 + u / fix_per_chunk, j = u % fix_per_chunk;
            const int need = (c - 1) * GPC + (j * kFixCols) / kGroup + 1;
            if (ld_acquire(sy + kSyGroups) >= need) {
                if (atomicCAS(sy + kSyUTicket, u, u + 1) == u) {
                    item[0] = kItemFix; item[1] = c; item[2] = j;
                    return;
                }
                continue;
            }
        }
        if (cur.ticket < 0) {
            cur.ticket = atomicAdd(sy + kSyTicket, 1);
            while (cur.c < a.nchunks && cur.ticket >= cur.base + normal_items(a.p.Np, C, a.nworkers, cur.c)) {
                cur.base += normal_items(a.p.Np, C, a.nworkers, cur.c);
                ++cur.c;
            }
        }
        if (cur.c >= a.nchunks) {           // normal queue exhausted
            if (u >= total_urgent) { item[0] = kItemExit; return; }
        } else if (cur.c < 2 || ld_acquire(sy + kSyGroups) >= (cur.c - 1) * GPC) {
            const int k = cur.ticket - cur.base;
            const int nd = diag_items(chunk_rows(a.p.Np, C, cur.c));
            item[0] = k < nd ? kItemDiag : kItemFar;
            item[1] = cur.c;
            item[2] = k < nd ? k : k - nd;
            cur.ticket = -1;
            return;
        }
        __nanosleep(200);
    }
}

template <int ROWS, bool UNIFORM>
__global__ void __launch_bounds__(kPThreads, 2) k_sweep(const PArgs a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    PShared& sh = *reinterpret_cast<PShared*>(smem_raw);
    const int tid = threadIdx.x, warp = tid >> 5;
    const Params& p = a.p;
    const int C = a.C;

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&sh.full_bar[s], 1);
            mbar_init(&sh.empty_bar[s], kBulkThreads / 32);
        }
        for (int s = 0; s < kRing; ++s) mbar_init(&sh.ho_bar[s], 2);
        for (int s = 0; s < 2 * (kChunkMax / kTile); ++s) mbar_init(&sh.a_bar[0][0] + s, 1);
        mbar_fence_init();
    }
    __syncthreads();

    if (blockIdx.x == 0) {
        chain_cta(a, sh);
        return;
    }

    Cursor cur{-1, 0, 0};
    unsigned kring = 0;
    for (;;) {
        __syncthreads();
        if (tid == 0) fetch_item(a, cur, sh.item);
        __syncthreads();
        const int type = sh.item[0], c = sh.item[1], k = sh.item[2];
        if (type == kItemExit) break;
        const int row0 = c * C, nrows = chunk_rows(p.Np, C, c);
        const ChunkBufs B = chunk_bufs(a, c);
        int* counter;
        if (type == kItemDiag) {
            if (warp < 8) {
                Params pc = p;
                pc.chunk = C;
                pc.partD = B.partD; pc.ovD = B.ovD; pc.Dblk = B.Dblk; pc.OVold = B.OVold; pc.OVnew = B.OVnew;
                diag_unit(pc, row0, nrows, k * 8 + warp, sh.u.w.cxy[warp], sh.u.w.czq[warp], sh.u.w.ctxy[warp],
                          sh.u.w.ch[warp], sh.u.w.ctz[warp]);
            }
            counter = sy_diag_done(a) + c;
        } else if (type == kItemFar) {
            const int prev0 = c > 0 ? row0 - C : row0;
            const int ncols = far_cols(p.Np, C, c);
            const int nf = far_slices(ncols, a.nworkers);
            const int v0 = slice_bound(ncols, nf, k), v1 = slice_bound(ncols, nf, k + 1);
            bulk_item<ROWS, UNIFORM>(p, sh, kring, row0, nrows, 0, p.Np, prev0, row0 + nrows, v0, v1,
                                     B.partA + (size_t)k * C, B.ovA + (size_t)k * C);
            counter = sy_far_done(a) + c;
        } else {
            const int cb = row0 - C + k * kFixCols;
            bulk_item<ROWS, UNIFORM>(p, sh, kring, row0, nrows, cb, cb + kFixCols, cb, cb, 0, kFixCols,
                                     B.partF + (size_t)k * C, B.ovF + (size_t)k * C);
            counter = sy_fix_done(a) + c;
        }
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            const int old = atomicAdd(counter, 1);
            __threadfence();
            sh.item[3] = old;
        }
        if (type != kItemFar) continue;
        __syncthreads();
        const int nf = far_slices(far_cols(p.Np, C, c), a.nworkers);
        if (sh.item[3] != nf - 1) continue;
        // last FAR item of the chunk: reduce the slots in a fixed order
        for (int r = tid; r < nrows; r += kPThreads) {
            double e[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            int ov = 0;
            for (int sl = 0; sl < nf; sl += 8) {
                double v[8];
                int o[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const bool in = sl + u < nf;
                    v[u] = in ? __ldcg(B.partA + (size_t)(sl + u) * C + r) : 0.0;
                    o[u] = in ? __ldcg(B.ovA + (size_t)(sl + u) * C + r) : 0;
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) { e[u] = __dadd_rn(e[u], v[u]); ov += o[u]; }
            }
            B.Efar[r] = __dadd_rn(__dadd_rn(__dadd_rn(e[0], e[1]), __dadd_rn(e[2], e[3])),
                                  __dadd_rn(__dadd_rn(e[4], e[5]), __dadd_rn(e[6], e[7])));
            B.ovfar[r] = ov;
        }
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            st_release(sy_far_ready(a) + c, 1);
        }
    }
}

}  // namespace mcb
