// kernels.cuh -- CUDA kernels of libmcb200 (sm_100a).  See DESIGN.md for the decomposition.
//
// One sweep = k_trial, then for every chunk of <= 1024 consecutive particles:
//   k_bulk   rows of the chunk x all columns outside the chunk, current positions   (a2)
//   k_diag   rows of the chunk x columns of the chunk: base sums at the chunk-start
//            positions plus, for every j < i, the correction D(i,j) that applies if j's
//            move is accepted, and the two overlap bit matrices                       (a2/a3)
//   k_chain  the sequential resolution: decisions in ascending i, D-corrections applied
//            as accept bits become known (ballot), commit of positions and log       (a3/a4)
// Because positions are committed in place chunk by chunk, "current positions" seen by
// k_bulk are x'_j for j before the chunk and x_j after it -- exactly Eq. 2.
#pragma once
#include "common.cuh"

namespace mcb {

struct Params {
    int N, Np, chunk;
    double2* xy;   // (x, y)  current positions                [Np]
    double2* zq;   // (z, q)                                   [Np]
    double* hh;    // d/2                                       [Np]
    double* lbq;   // l_B q                                     [Np]
    double2* txy;  // trial (x, y) of this sweep                [Np]
    double* tz;    // trial z                                   [Np]
    double* lnu;   // ln(u_acc)                                 [Np]
    unsigned char* wall;  // kFlagWall if vetoed by the wall    [Np]
    double* partA; int* ovA;   // [slices][chunk] partial sums / overlap counts of k_bulk
    double* partD; int* ovD;   // [chunk/32][chunk]              of k_diag
    double* Dblk;              // [nt(nt+1)/2][32 jj][32 ii] corrections, lower triangle of blocks
    unsigned* OVold; unsigned* OVnew;  // [chunk][chunk/32] bit jj of word s: trial i overlaps old/new j
    double* log_dE; unsigned char* log_flags;  // [Np]
    DevState* st;
    double R, lB, max_disp;
    unsigned long long seed;
    int* sy; int sy_n;         // scheduling state of the persistent sweep kernel (zeroed by k_trial)
    long long* S1; long long* S2; int* ovc;   // [Np] per-row fixed-point sums / overlap counts (persistent kernel)
    double* nn;                // [Np] |x_i|^2 of the current positions (persistent kernel's distance form)
};

// Order-independent accumulation of a row's partial sums (persistent kernel): the double is split
// exactly into a multiple of 2^-20 and a remainder below 2^-21 in magnitude, both added as 64-bit
// integers (the remainder in units of 2^-70: exact for |acc| >= 2^-18, else within 2^-71).  Integer
// addition is associative, so the total does not depend on which CTA adds first.  Range 2^43.
__device__ __forceinline__ void accum_row(const Params& p, int i, double acc, int ov) {
    const long long q1 = __double2ll_rn(__dmul_rn(acc, 0x1.0p20));
    const double rem = __fma_rn(__ll2double_rn(q1), -0x1.0p-20, acc);
    const long long q2 = __double2ll_rn(__dmul_rn(rem, 0x1.0p70));
    atomicAdd((unsigned long long*)(p.S1 + i), (unsigned long long)q1);
    atomicAdd((unsigned long long*)(p.S2 + i), (unsigned long long)q2);
    if (ov) atomicAdd(p.ovc + i, ov);
}
__device__ __forceinline__ double accum_value(long long s1, long long s2) {
    return __fma_rn(__ll2double_rn(s2), 0x1.0p-70, __dmul_rn(__ll2double_rn(s1), 0x1.0p-20));
}

// ------------------------------------------------------------------------------------------
// a1: trial generation.  Alg. 1 + old position (G1), D = 2 max_disp (G2),
// Philox keyed by (seed; particle, sweep, tag) (G9), hard wall (G6).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_trial(Params p) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    for (int j = i; j < p.sy_n; j += gridDim.x * blockDim.x) p.sy[j] = 0;
    if (i >= p.Np) return;
    p.S1[i] = 0ll; p.S2[i] = 0ll; p.ovc[i] = 0;
    const double2 xy = p.xy[i];
    const double2 zq = p.zq[i];
    if (i >= p.N) {  // ghost padding: never moves
        p.txy[i] = xy; p.tz[i] = zq.x; p.lnu[i] = 0.0; p.wall[i] = (unsigned char)kFlagWall;
        return;
    }
    const unsigned long long s = p.st->sweep;
    const uint32_t k0 = (uint32_t)p.seed, k1 = (uint32_t)(p.seed >> 32);
    uint32_t A[4], B[4];
    philox4x32_10((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 0u, k0, k1, A);
    philox4x32_10((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 1u, k0, k1, B);
    const double ux = uniform_open01(A[0], A[1]);
    const double uy = uniform_open01(A[2], A[3]);
    const double uz = uniform_open01(B[0], B[1]);
    const double ua = uniform_open01(B[2], B[3]);
    const double D = __dmul_rn(2.0, p.max_disp);
    const double tx = __fma_rn(__dadd_rn(ux, -0.5), D, xy.x);
    const double ty = __fma_rn(__dadd_rn(uy, -0.5), D, xy.y);
    const double tz = __fma_rn(__dadd_rn(uz, -0.5), D, zq.x);
    const double a = __dadd_rn(p.R, -p.hh[i]);
    const double rr = dist2(tx, ty, tz);
    p.txy[i] = make_double2(tx, ty);
    p.tz[i] = tz;
    p.lnu[i] = log(ua);
    p.wall[i] = (rr > __dmul_rn(a, a)) ? (unsigned char)kFlagWall : (unsigned char)0;
}

// ------------------------------------------------------------------------------------------
// a2: bulk pair energy.  Rows = trials of the chunk (one per consumer thread), columns = all
// particles outside [gap0, gap1) at their current positions, staged through shared memory by
// 1-D bulk async copies (TMA unit, mbarrier complete_tx) in a kStages ring.  Inner loop is the
// brush of Alg. 2: every lane reads the same column (smem broadcast).
// 27 FP64-pipe instructions + 2 MUFU.RSQ64H per pair evaluation.
// grid = (row groups, slices); block = kBulkRowsPerCta consumers + 1 producer warp.
// Partial sums go to slots slot0 .. slot0+nslices-1 of partA / ovA.
// ------------------------------------------------------------------------------------------
struct __align__(16) ColStage {
    double2 xy[kColTile];
    double2 zq[kColTile];
    double h[kColTile];
    double n[kColTile];
};

// slice boundaries in the virtual column space: multiples of 8, so that every staged segment
// holds a multiple of 8 columns (gap and range boundaries are multiples of 32) and the inner
// loop needs no tail
__host__ __device__ __forceinline__ int slice_bound(int ncols, int nslices, int sl) {
    return (int)(((long long)(ncols >> 3) * sl) / nslices) << 3;
}

// One pair evaluation (Eq. 2; Alg. 2): 22 FP64-pipe instructions
// (24 if diameters differ) + 2 MUFU.RSQ64H.
//   dx = x_i - x_j ...            3 DADD          r2o = fma(dz,dz,fma(dy,dy,dx dx))   3
//   w  = 2 D.(x_i - x_j) + |D|^2  3 DFMA          r2n = r2o + w                       1
//   (D = x~_i - x_i: |x~_i - x_j|^2 = |x_i - x_j|^2 + 2 D.(x_i - x_j) + |D|^2)
//   2 x rsqrt refinement          10              du, acc                             2
// The overlap veto is an integer test off the FP64 pipe: the running minimum of
// the high word of r2n (minus the high word of s_ij^2 if diameters differ).  r2n here is not in
// the evaluation order reading G11 fixes for the veto, so a row whose minimum falls within
// kOvBand high-word steps (2^-16 relative) of the threshold is re-examined exactly by
// recheck_overlap(); everything outside the band is decided by the minimum alone.
constexpr int kOvBand = 16;

struct RowRegs {
    double x, y, z;     // current position of the row's particle
    double ex, ey, ez;  // 2 (x~ - x)
    double c;           // |x~ - x|^2
    double h;           // d/2
    double acc;
    int m;              // running minimum of the overlap key
};

template <bool UNIFORM>
__device__ __forceinline__ int pair_eval(RowRegs& r, const double2 a, const double2 b, double hj) {
    const double dx = __dadd_rn(r.x, -a.x), dy = __dadd_rn(r.y, -a.y), dz = __dadd_rn(r.z, -b.x);
    const double r2o = dist2(dx, dy, dz);
    const double w = __fma_rn(r.ex, dx, __fma_rn(r.ey, dy, __fma_rn(r.ez, dz, r.c)));
    const double r2n = __dadd_rn(r2o, w);
    int key = __double2hiint(r2n);
    if (!UNIFORM) {
        const double sij = __dadd_rn(r.h, hj);
        key -= __double2hiint(__dmul_rn(sij, sij));
    }
    const double du = __dadd_rn(rsqrt_fast(r2n), -rsqrt_fast(r2o));
    r.acc = __fma_rn(b.y, du, r.acc);
    return key;
}

// Exact overlap test of trial i against the columns [v0, v1) of the virtual column space
// (reading G7/G11: r2 = fma(dz,dz,fma(dy,dy,dx dx)) of the rounded differences, strict <).
__device__ __noinline__ int recheck_overlap(const double2* xy, const double2* zq, const double* hh, double2 t,
                                            double tz, double hi, int v0, int v1, int cbeg, int gapv, int gap) {
    int ov = 0;
    for (int v = v0; v < v1; ++v) {
        const int j = cbeg + (v < gapv ? v : v + gap);
        const double2 a = xy[j];
        const double zj = zq[j].x;
        const double sij = __dadd_rn(hi, hh[j]);
        const double r2n = dist2(__dadd_rn(t.x, -a.x), __dadd_rn(t.y, -a.y), __dadd_rn(tz, -zj));
        ov |= (r2n < __dmul_rn(sij, sij)) ? 1 : 0;
    }
    return ov;
}

template <int ROWS, bool UNIFORM>
__global__ void __launch_bounds__(kBulkThreads + 32, ROWS == 1 ? 4 : 2)
k_bulk(Params p, int row0, int nrows, int cbeg, int cend, int gap0, int gap1, int nslices, int slot0) {
    __shared__ ColStage stage[kStages];
    __shared__ __align__(8) uint64_t full_bar[kStages];
    __shared__ __align__(8) uint64_t empty_bar[kStages];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int kConsumerWarps = kBulkThreads / 32;
    constexpr int kRowsPerCta = kBulkThreads * ROWS;
    // columns = [cbeg, cend) minus [gap0, gap1) (gap inside the range, or empty), as a virtual
    // index space v in [0, ncols): actual column = cbeg + v (+ gap if at or past the gap)
    const int gap = gap1 - gap0;
    const int ncols = (cend - cbeg) - gap;
    const int gapv = gap0 - cbeg;
    const int sl = blockIdx.y;
    const int v0 = slice_bound(ncols, nslices, sl), v1 = slice_bound(ncols, nslices, sl + 1);

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], kConsumerWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == kConsumerWarps) {
        // ---- producer: one lane walks the slice and feeds the ring ----
        if (lane == 0) {
            int k = 0;
            for (int v = v0; v < v1; ++k) {
                const int lim = (v < gapv) ? min(v1, gapv) : v1;
                const int cnt = min(kColTile, lim - v);
                const int a = cbeg + ((v < gapv) ? v : v + gap);
                const int s = k % kStages;
                if (k >= kStages) mbar_wait(&empty_bar[s], ((k / kStages) - 1) & 1);
                mbar_arrive_expect_tx(&full_bar[s], (uint32_t)cnt * (UNIFORM ? 32u : 40u));
                bulk_g2s(stage[s].xy, p.xy + a, (uint32_t)cnt * 16u, &full_bar[s]);
                bulk_g2s(stage[s].zq, p.zq + a, (uint32_t)cnt * 16u, &full_bar[s]);
                if (!UNIFORM) bulk_g2s(stage[s].h, p.hh + a, (uint32_t)cnt * 8u, &full_bar[s]);
                v += cnt;
            }
        }
        return;
    }

    // ---- consumers: ROWS rows per thread (row r, r + kBulkThreads, ...) ----
    const int rbase = blockIdx.x * kRowsPerCta;
    const bool warp_live = rbase + warp * 32 < nrows;   // whole warp past the chunk: only feed the barriers
    RowRegs R[ROWS];
#pragma unroll
    for (int u = 0; u < ROWS; ++u) {
        const int r = rbase + u * kBulkThreads + tid;
        const int i = row0 + (r < nrows ? r : 0);
        const double2 xyi = p.xy[i];
        const double2 txyi = p.txy[i];
        R[u].x = xyi.x; R[u].y = xyi.y; R[u].z = p.zq[i].x;
        const double Dx = __dadd_rn(txyi.x, -xyi.x), Dy = __dadd_rn(txyi.y, -xyi.y), Dz = __dadd_rn(p.tz[i], -R[u].z);
        R[u].ex = __dadd_rn(Dx, Dx); R[u].ey = __dadd_rn(Dy, Dy); R[u].ez = __dadd_rn(Dz, Dz);
        R[u].c = dist2(Dx, Dy, Dz);
        R[u].h = p.hh[i];
        R[u].acc = 0.0;
        R[u].m = 0x7fffffff;
    }

    int k = 0;
    for (int v = v0; v < v1; ++k) {
        const int lim = (v < gapv) ? min(v1, gapv) : v1;
        const int cnt = min(kColTile, lim - v);
        const int s = k % kStages;
        mbar_wait(&full_bar[s], (k / kStages) & 1);
        const ColStage& st = stage[s];
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
        if (lane == 0) mbar_arrive(&empty_bar[s]);
        v += cnt;
    }
#pragma unroll
    for (int u = 0; u < ROWS; ++u) {
        const int r = rbase + u * kBulkThreads + tid;
        // overlap key: high word of r2n relative to the high word of s^2
        int key = R[u].m;
        if (UNIFORM) {
            const double s = __dadd_rn(R[u].h, R[u].h);
            key -= __double2hiint(__dmul_rn(s, s));
        }
        int ov = key < 0 ? 1 : 0;
        if (r < nrows && key >= -kOvBand && key <= kOvBand)
            ov = recheck_overlap(p.xy, p.zq, p.hh, p.txy[row0 + r], p.tz[row0 + r], R[u].h, v0, v1, cbeg, gapv, gap);
        if (r < nrows) {
            p.partA[(size_t)(slot0 + sl) * p.chunk + r] = R[u].acc;
            p.ovA[(size_t)(slot0 + sl) * p.chunk + r] = ov;
        }
    }
}

// ------------------------------------------------------------------------------------------
// a2/a3 inside the chunk.  One warp per (row tile t, column tile s) of 32 x 32; lane = row.
//  s > t, or s == t and j > i : partner not yet decided when i is tried -> base term with x_j,
//                               overlap counted unconditionally.
//  s < t, or s == t and j < i : partner decided earlier in this chunk.  Base term with the
//                               chunk-start x_j (as if rejected) and D(i,j) = U(x~_j) - U(x_j)
//                               to add if j is accepted; overlap bits for both outcomes.
//    If the trial overlaps x_j the base term is dropped and D = U(x~_j) (i is vetoed anyway
//    unless j moves away); if it overlaps x~_j, D = 0 (i is vetoed if j is accepted).  So the
//    energy is exact whenever the trial is not vetoed and no inf/NaN enters a used sum.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int blk_index(int t, int s) { return t * (t + 1) / 2 + s; }

// one (row tile t, column tile s) unit, executed by one warp; the five arrays are this warp's
// 32-entry shared-memory staging rows
template <bool ATOMIC>
__device__ __forceinline__ void diag_unit(const Params& p, int row0, int nrows, int unit, double2* cxy, double2* czq,
                                          double2* ctxy, double* ch, double* ctz) {
    const int lane = threadIdx.x & 31;
    const int nt = nrows / kTile;
    if (unit >= nt * nt) return;
    const int t = unit / nt, s = unit % nt;
    const int r = t * kTile + lane, i = row0 + r;
    const int j0 = row0 + s * kTile;
    __syncwarp();
    cxy[lane] = p.xy[j0 + lane];
    czq[lane] = p.zq[j0 + lane];
    ctxy[lane] = p.txy[j0 + lane];
    ctz[lane] = p.tz[j0 + lane];
    ch[lane] = p.hh[j0 + lane];
    __syncwarp();
    const double2 xyi = p.xy[i];
    const double2 txyi = p.txy[i];
    const double xi = xyi.x, yi = xyi.y, zi = p.zq[i].x;
    const double txi = txyi.x, tyi = txyi.y, tzi = p.tz[i];
    const double hi = p.hh[i];
    const int W = p.chunk / kTile;
    double bsum = 0.0;
    int ovc = 0;
    unsigned ovo = 0u, ovn = 0u;
    double* blk = (s <= t) ? p.Dblk + (size_t)blk_index(t, s) * (kTile * kTile) : nullptr;
#pragma unroll 4
    for (int jj = 0; jj < kTile; ++jj) {
        const double2 a = cxy[jj];
        const double2 b = czq[jj];
        const double sij = __dadd_rn(hi, ch[jj]);
        const double s2 = __dmul_rn(sij, sij);
        const double r2oo = dist2(__dadd_rn(xi, -a.x), __dadd_rn(yi, -a.y), __dadd_rn(zi, -b.x));
        const double r2no = dist2(__dadd_rn(txi, -a.x), __dadd_rn(tyi, -a.y), __dadd_rn(tzi, -b.x));
        const bool upper = (s > t) || (s == t && jj > lane);
        const bool lower = (s < t) || (s == t && jj < lane);
        if (upper) {
            bsum = __fma_rn(b.y, __dadd_rn(rsqrt_fast(r2no), -rsqrt_fast(r2oo)), bsum);
            ovc += (r2no < s2) ? 1 : 0;
        } else if (lower) {
            const double2 ta = ctxy[jj];
            const double tzj = ctz[jj];
            const double r2on = dist2(__dadd_rn(xi, -ta.x), __dadd_rn(yi, -ta.y), __dadd_rn(zi, -tzj));
            const double r2nn = dist2(__dadd_rn(txi, -ta.x), __dadd_rn(tyi, -ta.y), __dadd_rn(tzi, -tzj));
            const bool oo = r2no < s2, on = r2nn < s2;
            double uold = 0.0, unew = 0.0;
            if (!oo) uold = __dmul_rn(b.y, __dadd_rn(rsqrt_fast(r2no), -rsqrt_fast(r2oo)));
            if (!on) unew = __dmul_rn(b.y, __dadd_rn(rsqrt_fast(r2nn), -rsqrt_fast(r2on)));
            bsum = __dadd_rn(bsum, uold);
            const double D = on ? 0.0 : __dadd_rn(unew, -uold);
            ovo |= (oo ? 1u : 0u) << jj;
            ovn |= (on ? 1u : 0u) << jj;
            blk[jj * kTile + lane] = D;
        } else {
            blk[jj * kTile + lane] = 0.0;  // jj == lane on the diagonal block
        }
        if (s == t && jj > lane) blk[jj * kTile + lane] = 0.0;
    }
    if (ATOMIC) {
        accum_row(p, i, bsum, ovc);
    } else {
        p.partD[(size_t)s * p.chunk + r] = bsum;
        p.ovD[(size_t)s * p.chunk + r] = ovc;
    }
    if (s <= t) {
        p.OVold[(size_t)r * W + s] = ovo;
        p.OVnew[(size_t)r * W + s] = ovn;
    }
}


__global__ void __launch_bounds__(256) k_diag(Params p, int row0, int nrows) {
    __shared__ double2 cxy[8][32], czq[8][32], ctxy[8][32];
    __shared__ double ch[8][32], ctz[8][32];
    const int w = threadIdx.x >> 5;
    diag_unit<false>(p, row0, nrows, blockIdx.x * 8 + w, cxy[w], czq[w], ctxy[w], ch[w], ctz[w]);
}

// ------------------------------------------------------------------------------------------
// a3/a4: sequential resolution of one chunk (Alg. 4).
// One CTA.  Warp 0 is the chain: lane l owns particle 32t+l of tile t; step j = lane j's
// decision, published by __ballot_sync; lanes > j add their precomputed D(l,j) if j accepted.
// While the chain resolves tile t, the other warps (a) add the corrections of the previous
// tile's accept mask A_{t-1} to the rows of tiles >= t+1 (block column t-1 of D, from L2) and
// (b) stage what the chain needs for tile t+1 in shared memory: the diagonal block (t+1,t+1),
// the block (t+1,t) -- applied by the chain warp itself as soon as A_t exists -- and the
// per-row scalars.  One __syncthreads per tile.
// accept iff no veto and l_B q_i sum + ln u < 0 (Eq. 1 in log form, strict; G3, G4).
// ------------------------------------------------------------------------------------------
constexpr int kChainThreads = 512;

struct ChainTileStage {
    double diag[kTile * kTile];   // D block (t, t)   [jj][lane]
    double prev[kTile * kTile];   // D block (t, t-1) [jj][lane]
    double lbq[kTile], lnu[kTile];
    unsigned ovoD[kTile], ovnD[kTile];  // overlap words of the diagonal block
    unsigned ovoP[kTile], ovnP[kTile];  // overlap words of block (t, t-1)
};

// Loads everything the chain needs for tile t into registers (issue phase) ...
struct ChainStageRegs {
    double d[5];
    double sc;
    unsigned w;
};

__device__ __forceinline__ void chain_stage_load(const Params& p, ChainStageRegs& rg, int row0, int t, int W,
                                                 int idx, int nthreads) {
    const double* dg = p.Dblk + (size_t)blk_index(t, t) * (kTile * kTile);
    const double* pv = p.Dblk + (size_t)blk_index(t, t > 0 ? t - 1 : 0) * (kTile * kTile);
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const int e = idx + k * nthreads;   // element of [diag | prev], 2048 in all
        rg.d[k] = 0.0;
        if (e < kTile * kTile) rg.d[k] = dg[e];
        else if (e < 2 * kTile * kTile && t > 0) rg.d[k] = pv[e - kTile * kTile];
    }
    const int a = idx >> 5, l = idx & 31, r = t * kTile + l;
    rg.sc = 0.0;
    rg.w = 0u;
    if (a == 0) rg.sc = p.lbq[row0 + r];
    else if (a == 1) rg.sc = p.lnu[row0 + r];
    else if (a == 2) rg.w = p.OVold[(size_t)r * W + t];
    else if (a == 3) rg.w = p.OVnew[(size_t)r * W + t];
    else if (a == 4 && t > 0) rg.w = p.OVold[(size_t)r * W + t - 1];
    else if (a == 5 && t > 0) rg.w = p.OVnew[(size_t)r * W + t - 1];
}

// ... and writes them to the shared stage (after the loads have been issued).
__device__ __forceinline__ void chain_stage_store(ChainTileStage& st, const ChainStageRegs& rg, int idx,
                                                  int nthreads) {
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const int e = idx + k * nthreads;
        if (e < kTile * kTile) st.diag[e] = rg.d[k];
        else if (e < 2 * kTile * kTile) st.prev[e - kTile * kTile] = rg.d[k];
    }
    const int a = idx >> 5, l = idx & 31;
    if (a == 0) st.lbq[l] = rg.sc;
    else if (a == 1) st.lnu[l] = rg.sc;
    else if (a == 2) st.ovoD[l] = rg.w;
    else if (a == 3) st.ovnD[l] = rg.w;
    else if (a == 4) st.ovoP[l] = rg.w;
    else if (a == 5) st.ovnP[l] = rg.w;
}

__global__ void __launch_bounds__(kChainThreads, 1)
k_chain(Params p, int row0, int nrows, int nslots, int last_chunk) {
    __shared__ double sE[kChunkMax];
    __shared__ unsigned char sVeto[kChunkMax];
    __shared__ ChainTileStage sT[2];
    __shared__ unsigned sA[kChunkMax / kTile];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int nwarps = kChainThreads / 32;
    const int nt = nrows / kTile;
    const int W = p.chunk / kTile;

    // prologue: reduce the partial sums in a fixed order (16 independent accumulators per row,
    // combined in a fixed tree, so the result does not depend on scheduling)
    for (int r = tid; r < nrows; r += kChainThreads) {
        double e[16];
        int ov = 0;
#pragma unroll
        for (int u = 0; u < 16; ++u) e[u] = 0.0;
        for (int sl = 0; sl < nslots; sl += 16) {
            double v[16];
            int o[16];
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                const bool in = sl + u < nslots;
                v[u] = in ? p.partA[(size_t)(sl + u) * p.chunk + r] : 0.0;
                o[u] = in ? p.ovA[(size_t)(sl + u) * p.chunk + r] : 0;
            }
#pragma unroll
            for (int u = 0; u < 16; ++u) { e[u] += v[u]; ov += o[u]; }
        }
        for (int s0 = 0; s0 < nt; s0 += 16) {
            double v[16];
            int o[16];
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                const bool in = s0 + u < nt;
                v[u] = in ? p.partD[(size_t)(s0 + u) * p.chunk + r] : 0.0;
                o[u] = in ? p.ovD[(size_t)(s0 + u) * p.chunk + r] : 0;
            }
#pragma unroll
            for (int u = 0; u < 16; ++u) { e[u] += v[u]; ov += o[u]; }
        }
#pragma unroll
        for (int w = 8; w > 0; w >>= 1)
#pragma unroll
            for (int u = 0; u < w; ++u) e[u] += e[u + w];
        sE[r] = e[0];
        sVeto[r] = (unsigned char)(p.wall[row0 + r] | (ov > 0 ? kFlagOverlap : 0u));
    }
    {
        ChainStageRegs rg;
        chain_stage_load(p, rg, row0, 0, W, tid, kChainThreads);
        chain_stage_store(sT[0], rg, tid, kChainThreads);
    }
    __syncthreads();

    unsigned long long n_acc = 0, n_ov = 0, n_wall = 0, n_tie = 0;
    double e_run = 0.0;

    for (int t = 0; t < nt; ++t) {
        if (warp == 0) {
            // ---------------- the chain ----------------
            const ChainTileStage& st = sT[t & 1];
            const int r = t * kTile + lane, i = row0 + r;
            const double lbq = st.lbq[lane], lnu = st.lnu[lane];
            double Eu = sE[r];
            const unsigned vflags = sVeto[r];
            const bool wallv = (vflags & kFlagWall) != 0u;
            bool ovv = (vflags & kFlagOverlap) != 0u;
            if (t > 0) {  // corrections of the tile just resolved (block (t, t-1))
                const unsigned Ap = sA[t - 1];
#pragma unroll
                for (int jj = 0; jj < kTile; ++jj)
                    if ((Ap >> jj) & 1u) Eu = __dadd_rn(Eu, st.prev[jj * kTile + lane]);
                ovv = ovv || (((st.ovnP[lane] & Ap) | (st.ovoP[lane] & ~Ap)) != 0u);
            }
            double Es = __fma_rn(lbq, Eu, lnu);
            const unsigned ovo = st.ovoD[lane], ovn = st.ovnD[lane];
            unsigned A = 0u;
#pragma unroll
            for (int j = 0; j < kTile; ++j) {
                const double dj = st.diag[j * kTile + lane];   // 0 for lanes <= j
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
            if (lane == 0) sA[t] = A;
            const bool acc = ((A >> lane) & 1u) != 0u;
            const double dE = __dmul_rn(lbq, Eu);
            const bool tie = !wallv && !ovv && (fabs(Es) < 1e-8);
            if (acc) {
                const double2 txy = p.txy[i];
                const double tz = p.tz[i];
                const double q = p.zq[i].y;
                p.xy[i] = txy;
                p.zq[i] = make_double2(tz, q);
                p.nn[i] = dist2(txy.x, txy.y, tz);
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
        } else {
            // ---------------- helpers ----------------
            const int hid = tid - 32;
            constexpr int nh = kChainThreads - 32;
            const unsigned Ap = t > 0 ? sA[t - 1] : 0u;
            // issue: corrections of mask A_{t-1} for the first far tile of this warp ...
            int t2 = t + warp;   // tiles t+1 .. nt-1, round-robin over the helper warps
            double v[kTile];
            const bool far0 = t > 0 && t2 < nt;
            {
                const double* blk = p.Dblk + (size_t)blk_index(far0 ? t2 : 1, far0 ? t - 1 : 0) * (kTile * kTile);
#pragma unroll
                for (int jj = 0; jj < kTile; ++jj)
                    v[jj] = (far0 && ((Ap >> jj) & 1u)) ? blk[jj * kTile + lane] : 0.0;
            }
            // ... and everything the chain needs for tile t+1
            ChainStageRegs rg;
            const bool stage = t + 1 < nt;
            if (stage) chain_stage_load(p, rg, row0, t + 1, W, hid, nh);
            if (stage) chain_stage_store(sT[(t + 1) & 1], rg, hid, nh);
            // consume
            bool first = true;
            for (; t > 0 && t2 < nt; t2 += nwarps - 1) {
                const int r = t2 * kTile + lane;
                if (!first) {
                    const double* blk = p.Dblk + (size_t)blk_index(t2, t - 1) * (kTile * kTile);
#pragma unroll
                    for (int jj = 0; jj < kTile; ++jj) v[jj] = ((Ap >> jj) & 1u) ? blk[jj * kTile + lane] : 0.0;
                }
                first = false;
                const unsigned on = p.OVnew[(size_t)r * W + t - 1], oo = p.OVold[(size_t)r * W + t - 1];
                double s4[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
                for (int jj = 0; jj < kTile; ++jj) s4[jj & 3] = __dadd_rn(s4[jj & 3], v[jj]);
                sE[r] = __dadd_rn(sE[r], __dadd_rn(__dadd_rn(s4[0], s4[1]), __dadd_rn(s4[2], s4[3])));
                if (((on & Ap) | (oo & ~Ap)) != 0u) sVeto[r] |= (unsigned char)kFlagOverlap;
            }
        }
        __syncthreads();
    }
    if (tid == 0) {
        DevState* st = p.st;
        st->accepted += n_acc;
        st->veto_overlap += n_ov;
        st->veto_wall += n_wall;
        st->near_ties += n_tie;
        st->E_run += e_run;
        if (last_chunk) st->sweep += 1ull;
    }
}

// ------------------------------------------------------------------------------------------
// packing between the caller's SoA [3][N] and the workspace layout
// ------------------------------------------------------------------------------------------
__global__ void k_pack(Params p, const double* pos, const double* q, const double* d) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.Np) return;
    if (i < p.N) {
        p.xy[i] = make_double2(pos[i], pos[(size_t)p.N + i]);
        p.nn[i] = dist2(pos[i], pos[(size_t)p.N + i], pos[2 * (size_t)p.N + i]);
        if (q) {
            p.zq[i] = make_double2(pos[2 * (size_t)p.N + i], q[i]);
            p.hh[i] = __dmul_rn(0.5, d[i]);
            p.lbq[i] = __dmul_rn(p.lB, q[i]);
        } else {
            p.zq[i].x = pos[2 * (size_t)p.N + i];
        }
    } else if (q) {
        p.xy[i] = make_double2(kGhostCoord + kGhostStep * (double)(i - p.N), 0.0);
        p.nn[i] = __dmul_rn(kGhostCoord + kGhostStep * (double)(i - p.N), kGhostCoord + kGhostStep * (double)(i - p.N));
        p.zq[i] = make_double2(0.0, 0.0);
        p.hh[i] = 0.0;
        p.lbq[i] = 0.0;
    }
}

__global__ void k_unpack(Params p, double* pos) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.N) return;
    const double2 xy = p.xy[i];
    pos[i] = xy.x;
    pos[(size_t)p.N + i] = xy.y;
    pos[2 * (size_t)p.N + i] = p.zq[i].x;
}

__global__ void k_set_sweep(DevState* st, unsigned long long s) { st->sweep = s; }

__global__ void k_copy_log(Params p, double* dE, unsigned char* flags) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.N) return;
    if (dE) dE[i] = p.log_dE[i];
    if (flags) flags[i] = p.log_flags[i];
}

// per-particle input checks: finite, d > 0, inside the wall
__global__ void k_check_particles(Params p, const double* d) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.N) return;
    const double2 xy = p.xy[i];
    const double2 zq = p.zq[i];
    const double di = d[i];
    int err = 0;
    if (!isfinite(xy.x) || !isfinite(xy.y) || !isfinite(zq.x) || !isfinite(zq.y) || !isfinite(di) ||
        !(di > 0.0)) {
        err = -1;
    } else {
        const double a = __dadd_rn(p.R, -p.hh[i]);
        if (!(a >= 0.0) || dist2(xy.x, xy.y, zq.x) > __dmul_rn(a, a)) err = -3;
    }
    if (err) atomicMin(&p.st->err, err == -1 ? -1000 : err);  // EINVAL outranks the others
    if (di != d[0]) p.st->d_differs = 1;
    if (di > 0.0) atomicMin(&p.st->dmin_bits, (unsigned long long)__double_as_longlong(di));   // positive doubles order as integers
}

// ------------------------------------------------------------------------------------------
// a5: from-scratch energy (and the overlap check of mc_init): E = l_B sum_{i<j} q_i q_j / r_ij.
// The upper triangle is cut into units of 1024 rows x 1024 columns (4 column tiles of 256); one CTA
// per unit, 4 rows per thread, columns staged through shared memory, 10 FP64-pipe instructions per
// pair.  Units on the diagonal test j > i per pair.  Every CTA reduces its rows in a fixed order and
// writes one partial; k_energy_reduce adds the partials in index order.
// ------------------------------------------------------------------------------------------
constexpr int kERows = 4, kEBlock = 256 * kERows, kETile = 256;

__host__ __device__ inline int energy_units(int Np) {
    const int nrb = (Np + kEBlock - 1) / kEBlock;
    int n = 0;
    for (int rb = 0; rb < nrb; ++rb) n += ((Np - rb * kEBlock) + kEBlock - 1) / kEBlock;
    return n;
}

template <bool CHECK>
__global__ void __launch_bounds__(256, 2) k_energy(Params p, double* part) {
    __shared__ double2 sxy[kETile], szq[kETile];
    __shared__ double sh[kETile], sn[kETile];
    __shared__ double red[8];
    const int tid = threadIdx.x;
    // unit -> (row block rb, column block cb >= rb)
    int unit = blockIdx.x, rb = 0;
    for (;;) {
        const int n = ((p.Np - rb * kEBlock) + kEBlock - 1) / kEBlock;
        if (unit < n) break;
        unit -= n;
        ++rb;
    }
    const int cb = rb + unit;
    // off the diagonal: r^2 = |x_i|^2 + |x_j|^2 - 2 x_i.x_j (1 DADD + 3 DFMA; |x|^2 is kept per particle, p.nn),
    // 10 FP64-pipe instructions per pair; on the diagonal and in the overlap check of mc_init the
    // differences are formed explicitly (reading G11's evaluation order)
    double x[kERows], y[kERows], z[kERows], q[kERows], h[kERows], nn[kERows], acc[kERows];
    int bad = 0;
#pragma unroll
    for (int u = 0; u < kERows; ++u) {
        const int i = rb * kEBlock + u * 256 + tid;
        const bool live = i < p.Np;
        const double2 xy = live ? p.xy[i] : make_double2(3.0e9, 0.0);
        const double2 zq = live ? p.zq[i] : make_double2(0.0, 0.0);
        x[u] = xy.x; y[u] = xy.y; z[u] = zq.x; q[u] = zq.y;
        h[u] = live ? p.hh[i] : 0.0;
        nn[u] = live ? p.nn[i] : 9.0e18;
        acc[u] = 0.0;
    }
    const bool diagonal = cb == rb;
    double mx[kERows], my[kERows], mz[kERows];
#pragma unroll
    for (int u = 0; u < kERows; ++u) { mx[u] = __dmul_rn(-2.0, x[u]); my[u] = __dmul_rn(-2.0, y[u]); mz[u] = __dmul_rn(-2.0, z[u]); }
    for (int ct = 0; ct < kEBlock / kETile; ++ct) {
        const int j0 = cb * kEBlock + ct * kETile;
        if (j0 >= p.Np) break;
        const int cnt = min(kETile, p.Np - j0);
        __syncthreads();
        if (tid < cnt) {
            sxy[tid] = p.xy[j0 + tid]; szq[tid] = p.zq[j0 + tid]; sn[tid] = p.nn[j0 + tid];
            if (CHECK) sh[tid] = p.hh[j0 + tid];
        }
        __syncthreads();
        if (!diagonal && !CHECK) {
#pragma unroll 2
            for (int j = 0; j < cnt; ++j) {
                const double2 a = sxy[j], b = szq[j];
                const double nj = sn[j];
#pragma unroll
                for (int u = 0; u < kERows; ++u) {
                    const double r2 = __fma_rn(mx[u], a.x, __fma_rn(my[u], a.y, __fma_rn(mz[u], b.x, __dadd_rn(nn[u], nj))));
                    acc[u] = __fma_rn(b.y, rsqrt_fast(r2), acc[u]);
                }
            }
        } else {
            for (int j = 0; j < cnt; ++j) {
                const double2 a = sxy[j], b = szq[j];
#pragma unroll
                for (int u = 0; u < kERows; ++u) {
                    const int i = rb * kEBlock + u * 256 + tid;
                    if (j0 + j > i) {
                        const double r2 = dist2(__dadd_rn(x[u], -a.x), __dadd_rn(y[u], -a.y), __dadd_rn(z[u], -b.x));
                        acc[u] = __fma_rn(b.y, rsqrt_fast(r2), acc[u]);
                        if (CHECK) {
                            const double sij = __dadd_rn(h[u], sh[j]);
                            bad |= (r2 < __dmul_rn(sij, sij)) && (j0 + j < p.N) && (i < p.N);
                        }
                    }
                }
            }
        }
    }
    // fixed-order reduction: rows of the thread, lanes of the warp, warps of the CTA
    double v = 0.0;
#pragma unroll
    for (int u = 0; u < kERows; ++u) v = __dadd_rn(v, __dmul_rn(q[u], acc[u]));
    v = warp_sum(v);
    if ((tid & 31) == 0) red[tid >> 5] = v;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t = __dadd_rn(t, red[w]);
        part[blockIdx.x] = t;
    }
    if (bad) atomicMin(&p.st->err, -2);
}

// out = l_B * sum of the partials in index order (one warp; lane l adds partials l, l+32, ...)
__global__ void __launch_bounds__(32) k_energy_reduce(Params p, const double* part, int nparts, double* out,
                                                      int set_running) {
    double acc = 0.0;
    for (int k = threadIdx.x; k < nparts; k += 32) acc = __dadd_rn(acc, part[k]);
    acc = warp_sum(acc);
    if (threadIdx.x == 0) {
        const double E = __dmul_rn(p.lB, acc);
        if (out) *out = E;
        if (set_running) p.st->E_run = E;
    }
}

// ------------------------------------------------------------------------------------------
// a6: pair-distance histograms.  k_centres lists the bulk ions in
// index order; k_hist bins (centre, any partner) distances into shared-memory histograms.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_centres(Params p, double centre_rmax, int* list, int* count,
                                                  unsigned long long* n_centres) {
    __shared__ int wcount[32];
    __shared__ int base;
    __shared__ unsigned long long nsp[2];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) { base = 0; nsp[0] = nsp[1] = 0ull; }
    __syncthreads();
    const double c2 = __dmul_rn(centre_rmax, centre_rmax);
    for (int i0 = 0; i0 < p.N; i0 += 1024) {
        const int i = i0 + tid;
        bool is = false;
        int sp = 0;
        if (i < p.N) {
            const double2 xy = p.xy[i];
            const double2 zq = p.zq[i];
            is = dist2(xy.x, xy.y, zq.x) <= c2;
            sp = zq.y > 0.0 ? 0 : 1;
        }
        const unsigned m = __ballot_sync(0xffffffffu, is);
        const unsigned m0 = __ballot_sync(0xffffffffu, is && sp == 0);
        if (lane == 0) wcount[warp] = __popc(m);
        __syncthreads();
        int off = base;
        for (int w = 0; w < warp; ++w) off += wcount[w];
        if (is) list[off + __popc(m & ((1u << lane) - 1u))] = i;
        if (lane == 0) {
            atomicAdd(&nsp[0], (unsigned long long)__popc(m0));
            atomicAdd(&nsp[1], (unsigned long long)(__popc(m) - __popc(m0)));
        }
        __syncthreads();
        if (tid == 0) {
            int tot = 0;
            for (int w = 0; w < 32; ++w) tot += wcount[w];
            base += tot;
        }
        __syncthreads();
    }
    if (tid == 0) {
        *count = base;
        n_centres[0] += nsp[0];
        n_centres[1] += nsp[1];
    }
}

constexpr int kHistSlices = 32;
constexpr int kCellBits = 4, kCellDim = 1 << kCellBits, kCells = 1 << (3 * kCellBits);

// The partners of a centre within nbins * bin_width are found through a spatially sorted copy of
// the configuration: particles are counting-sorted by the Morton code of their cell (k_cell_*), so
// that 256 consecutive particles fill a compact box; k_hist takes 256 consecutive centres and skips
// every 256-particle column tile whose bounding box is farther than the histogram's range from the
// centres' bounding box.  The counts do not depend on the order inside a cell (integer adds).
struct CellGrid {
    double lo, inv_edge;   // cell coordinate = clamp(floor((x - lo) * inv_edge), 0, dim - 1)
    int dim;
};
__device__ __forceinline__ unsigned spread5(unsigned v) {   // dcba -> d00c00b00a
    return (v & 1u) | ((v & 2u) << 2) | ((v & 4u) << 4) | ((v & 8u) << 6);
}
__device__ __forceinline__ int cell_code(const CellGrid& g, double x, double y, double z) {
    const int cx = min(g.dim - 1, max(0, (int)floor((x - g.lo) * g.inv_edge)));
    const int cy = min(g.dim - 1, max(0, (int)floor((y - g.lo) * g.inv_edge)));
    const int cz = min(g.dim - 1, max(0, (int)floor((z - g.lo) * g.inv_edge)));
    return (int)(spread5((unsigned)cx) | (spread5((unsigned)cy) << 1) | (spread5((unsigned)cz) << 2));
}
__global__ void __launch_bounds__(256) k_cell_count(Params p, CellGrid g, int* code, int* count) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.N) return;
    const double2 xy = p.xy[i];
    const int c = cell_code(g, xy.x, xy.y, p.zq[i].x);
    code[i] = c;
    atomicAdd(count + c, 1);
}
// exclusive scan of count[kCells] into cursor[kCells]; one CTA of 1024 threads, 32 cells each
__global__ void __launch_bounds__(1024) k_cell_scan(const int* count, int* cursor) {
    __shared__ int wsum[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int per = kCells / 1024;
    int loc[per], tot = 0;
#pragma unroll
    for (int k = 0; k < per; ++k) { loc[k] = tot; tot += count[tid * per + k]; }
    int inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        int w = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o) w += v;
        }
        wsum[lane] = w;
    }
    __syncthreads();
    const int base = inc - tot + (warp > 0 ? wsum[warp - 1] : 0);
#pragma unroll
    for (int k = 0; k < per; ++k) cursor[tid * per + k] = base + loc[k];
}
__global__ void __launch_bounds__(256) k_cell_fill(Params p, const int* code, int* cursor, double2* sxy, double2* szq) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.N) return;
    const int pos = atomicAdd(cursor + code[i], 1);
    sxy[pos] = p.xy[i];
    szq[pos] = p.zq[i];
}
// bounding box of every sub-tile of 64 consecutive sorted particles: bbox[t] = {xmin, xmax, ymin, ymax, zmin, zmax}
constexpr int kSubTile = 64;
__global__ void __launch_bounds__(256) k_tile_bbox(const double2* sxy, const double2* szq, int N, double* bbox) {
    const int tid = threadIdx.x, j = blockIdx.x * 256 + tid;
    double v[6] = {1e300, -1e300, 1e300, -1e300, 1e300, -1e300};
    if (j < N) {
        const double2 a = sxy[j];
        const double z = szq[j].x;
        v[0] = v[1] = a.x; v[2] = v[3] = a.y; v[4] = v[5] = z;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const double w = __shfl_xor_sync(0xffffffffu, v[k], o);
            v[k] = (k & 1) ? fmax(v[k], w) : fmin(v[k], w);
        }
    __shared__ double red[8][6];
    if ((tid & 31) == 0)
        for (int k = 0; k < 6; ++k) red[tid >> 5][k] = v[k];
    __syncthreads();
    if (tid < 24) {   // 4 sub-tiles x 6 values, each from 2 warps
        const int st = tid / 6, k = tid % 6;
        const double a = red[2 * st][k], b = red[2 * st + 1][k];
        bbox[((size_t)blockIdx.x * 4 + st) * 6 + k] = (k & 1) ? fmax(a, b) : fmin(a, b);
    }
}

// centres (|x_i| <= centre_rmax) of the sorted copy, compacted per 1024-particle block (blocks land
// in the list in completion order, each block's centres stay together and in order)
__global__ void __launch_bounds__(1024) k_centres_sorted(Params p, double centre_rmax, int* list, int* count,
                                                         unsigned long long* n_centres) {
    __shared__ int wcount[32];
    __shared__ int base;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int i = blockIdx.x * 1024 + tid;
    const double c2 = __dmul_rn(centre_rmax, centre_rmax);
    bool is = false;
    int sp = 0;
    if (i < p.N) {
        const double2 xy = p.xy[i];
        const double2 zq = p.zq[i];
        is = dist2(xy.x, xy.y, zq.x) <= c2;
        sp = zq.y > 0.0 ? 0 : 1;
    }
    const unsigned m = __ballot_sync(0xffffffffu, is);
    const unsigned m0 = __ballot_sync(0xffffffffu, is && sp == 0);
    if (lane == 0) {
        wcount[warp] = __popc(m);
        if (m0) atomicAdd(n_centres + 0, (unsigned long long)__popc(m0));
        if (m & ~m0) atomicAdd(n_centres + 1, (unsigned long long)__popc(m & ~m0));
    }
    __syncthreads();
    if (tid == 0) {
        int tot = 0;
        for (int w = 0; w < 32; ++w) { const int c = wcount[w]; wcount[w] = tot; tot += c; }
        base = tot ? atomicAdd(count, tot) : 0;
    }
    __syncthreads();
    if (is) list[base + wcount[warp] + __popc(m & ((1u << lane) - 1u))] = i;
}

// p.xy / p.zq here are the SORTED copies; list = sorted indices of the centres
__global__ void __launch_bounds__(256) k_hist(Params p, const int* list, const int* count, const double* bbox,
                                              double inv_w, int nbins, double cut2, unsigned long long* hist) {
    extern __shared__ unsigned shist[];  // [4][nbins]
    __shared__ double2 sxy[256], szq[256];
    __shared__ double cred[8][6];
    __shared__ double cbox[6];
    const int tid = threadIdx.x;
    const int nc = *count;
    if ((int)blockIdx.x * 256 >= nc) return;
    for (int b = tid; b < 4 * nbins; b += 256) shist[b] = 0u;
    const int c = blockIdx.x * 256 + tid;
    const bool live = c < nc;
    const int i = live ? list[c] : -1;
    double2 xyi = make_double2(0, 0), zqi = make_double2(0, 0);
    if (live) { xyi = p.xy[i]; zqi = p.zq[i]; }
    const int si = zqi.y > 0.0 ? 0 : 1;
    // bounding box of this block's centres
    {
        double v[6] = {1e300, -1e300, 1e300, -1e300, 1e300, -1e300};
        if (live) { v[0] = v[1] = xyi.x; v[2] = v[3] = xyi.y; v[4] = v[5] = zqi.x; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const double w = __shfl_xor_sync(0xffffffffu, v[k], o);
                v[k] = (k & 1) ? fmax(v[k], w) : fmin(v[k], w);
            }
        if ((tid & 31) == 0)
            for (int k = 0; k < 6; ++k) cred[tid >> 5][k] = v[k];
        __syncthreads();
        if (tid < 6) {
            double r = cred[0][tid];
            for (int w = 1; w < 8; ++w) r = (tid & 1) ? fmax(r, cred[w][tid]) : fmin(r, cred[w][tid]);
            cbox[tid] = r;
        }
        __syncthreads();
    }
    const int ntile = (p.N + 255) / 256;
    const double margin = 1.0 + 1e-6;   // the cull is conservative: only tiles clearly out of range are skipped
    for (int ct = blockIdx.y; ct < ntile; ct += gridDim.y) {
        // which of the tile's 4 sub-tiles of 64 are in range of this block's centres (same in every thread)
        unsigned inrange = 0u;
#pragma unroll
        for (int st = 0; st < 4; ++st) {
            const double* bb = bbox + ((size_t)ct * 4 + st) * 6;
            double d2 = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double gap = fmax(0.0, fmax(bb[2 * k] - cbox[2 * k + 1], cbox[2 * k] - bb[2 * k + 1]));
                d2 += gap * gap;
            }
            if (d2 <= cut2 * margin) inrange |= 1u << st;
        }
        if (inrange == 0u) continue;
        const int j0 = ct * 256;
        __syncthreads();
        if (j0 + tid < p.N) { sxy[tid] = p.xy[j0 + tid]; szq[tid] = p.zq[j0 + tid]; }
        __syncthreads();
        const int cnt = min(256, p.N - j0);
        if (!live) continue;
        for (int st = 0; st < 4; ++st) {
            if (!((inrange >> st) & 1u)) continue;
            const int jend = min(cnt, (st + 1) * kSubTile);
#pragma unroll 4
            for (int j = st * kSubTile; j < jend; ++j) {
                const double2 a = sxy[j], b = szq[j];
                const double r2 = dist2(__dadd_rn(xyi.x, -a.x), __dadd_rn(xyi.y, -a.y), __dadd_rn(zqi.x, -b.x));
                if (r2 < cut2 && (j0 + j) != i) {
                    const double fb = floor(__dmul_rn(sqrt(r2), inv_w));
                    if (fb < (double)nbins) {
                        const int sj = b.y > 0.0 ? 0 : 1;
                        atomicAdd(&shist[(si * 2 + sj) * nbins + (int)fb], 1u);
                    }
                }
            }
        }
    }
    __syncthreads();
    for (int b = tid; b < 4 * nbins; b += 256) {
        const unsigned v = shist[b];
        if (v) atomicAdd(&hist[b], (unsigned long long)v);
    }
}

// ------------------------------------------------------------------------------------------
// FP64 peak probe: 8 independent DFMA chains per thread, register resident.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_dfma_peak(double* sink, int iters) {
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6,
           a7 = a0 + 7;
    const double m = 1.0000001, c = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = __fma_rn(a0, m, c); a1 = __fma_rn(a1, m, c); a2 = __fma_rn(a2, m, c); a3 = __fma_rn(a3, m, c);
            a4 = __fma_rn(a4, m, c); a5 = __fma_rn(a5, m, c); a6 = __fma_rn(a6, m, c); a7 = __fma_rn(a7, m, c);
        }
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123.456) sink[0] = s;
}

}  // namespace mcb
