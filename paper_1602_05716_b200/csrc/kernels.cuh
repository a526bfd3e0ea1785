// kernels.cuh -- device code shared by the sweep kernel (persist.cuh) and the kernels around it
// (aux_kernels.cuh): the workspace view, the order-independent row accumulators, the column stage of
// the pair loop and the speculative in-chunk unit (a2/a3).  sm_100a only.  See DESIGN.md.
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
    double* Dblk;              // [nt(nt+1)/2][32 jj][32 ii] corrections, lower triangle of blocks
    unsigned* OVold; unsigned* OVnew;  // [chunk][chunk/32] bit jj of word s: trial i overlaps old/new j
    double* log_dE; unsigned char* log_flags;  // [Np]
    DevState* st;
    double R, lB, max_disp;
    unsigned long long seed;
    int* sy; int sy_n;         // scheduling state of the sweep kernel (zero between sweeps)
    long long* S1; long long* S2; int* ovc;   // [Np] per-row fixed-point sums / overlap counts (persistent kernel)
    double* nn;                // [Np] |x_i|^2 of the current positions (Gram form of the pair distance)
    double ov_tol;             // half-width of the band around contact inside which a veto is re-examined exactly
    unsigned long long wait_limit_ns;   // watchdog limit per wait of the sweep kernel (0: none)
    int pos_bits;              // 64, or 32: every position the chain holds is an FP32 value, arithmetic stays FP64
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
// a1: trial generation for particle i of sweep s.  Alg. 1 + old position (G1), D = 2 max_disp
// (G2), Philox keyed by (seed; particle, sweep, tag) (G9), hard wall (G6).  Also clears the row's
// accumulators.  Runs inside the sweep kernel (persist.cuh: trial_phase), all threads of the grid.
// ------------------------------------------------------------------------------------------
struct Trial {
    double x, y, z, lnu;
    unsigned char wall;
};
__device__ __forceinline__ Trial trial_compute(const Params& p, int i, unsigned long long s, double2 xy, double zi) {
    const uint32_t k0 = (uint32_t)p.seed, k1 = (uint32_t)(p.seed >> 32);
    uint32_t A[4], B[4];
    philox4x32_10((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 0u, k0, k1, A);
    philox4x32_10((uint32_t)i, (uint32_t)s, (uint32_t)(s >> 32), 1u, k0, k1, B);
    const double ux = uniform_open01(A[0], A[1]);
    const double uy = uniform_open01(A[2], A[3]);
    const double uz = uniform_open01(B[0], B[1]);
    const double ua = uniform_open01(B[2], B[3]);
    const double D = __dmul_rn(2.0, p.max_disp);
    Trial t;
    t.x = __fma_rn(__dadd_rn(ux, -0.5), D, xy.x);
    t.y = __fma_rn(__dadd_rn(uy, -0.5), D, xy.y);
    t.z = __fma_rn(__dadd_rn(uz, -0.5), D, zi);
    if (p.pos_bits == 32) {   // the proposed position is stored as FP32: one more rounding, to nearest
        t.x = (double)__double2float_rn(t.x); t.y = (double)__double2float_rn(t.y); t.z = (double)__double2float_rn(t.z);
    }
    const double a = __dadd_rn(p.R, -p.hh[i]);
    const double rr = dist2(t.x, t.y, t.z);
    t.lnu = log(ua);
    t.wall = (rr > __dmul_rn(a, a)) ? (unsigned char)kFlagWall : (unsigned char)0;
    return t;
}
__device__ __forceinline__ void trial_one(const Params& p, int i, unsigned long long s) {
    p.S1[i] = 0ll; p.S2[i] = 0ll; p.ovc[i] = 0;
    const double2 xy = p.xy[i];
    const double2 zq = p.zq[i];
    if (i >= p.N) {  // ghost padding: never moves
        p.txy[i] = xy; p.tz[i] = zq.x; p.lnu[i] = 0.0; p.wall[i] = (unsigned char)kFlagWall;
        return;
    }
    const Trial t = trial_compute(p, i, s, xy, zq.x);
    p.txy[i] = make_double2(t.x, t.y);
    p.tz[i] = t.z;
    p.lnu[i] = t.lnu;
    p.wall[i] = t.wall;
}

// ------------------------------------------------------------------------------------------
// a2: bulk pair energy -- what the sweep kernel stages per column (persist.cuh holds the pair loop).
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
// Columns jj0 <= jj < jj1 of the unit only: several warps may share a unit (the multi-thread-per-particle idea of
// the terms of one trial spread over eta "slave" threads when the system is too small to
// fill the device); ovo / ovn return this part's overlap bits, which the caller combines over the parts.
__device__ __forceinline__ void diag_unit(const Params& p, int row0, int nrows, int unit, double2* cxy, double2* czq,
                                          double2* ctxy, double* ch, double* ctz, int jj0, int jj1, unsigned& ovo_out,
                                          unsigned& ovn_out) {
    const int lane = threadIdx.x & 31;
    const int nt = nrows / kTile;
    ovo_out = 0u; ovn_out = 0u;
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
    double bsum = 0.0;
    int ovc = 0;
    unsigned ovo = 0u, ovn = 0u;
    double* blk = (s <= t) ? p.Dblk + (size_t)blk_index(t, s) * (kTile * kTile) : nullptr;
#pragma unroll 4
    for (int jj = jj0; jj < jj1; ++jj) {
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
    accum_row(p, i, bsum, ovc);
    ovo_out = ovo; ovn_out = ovn;
}


}  // namespace mcb
