// common.cuh -- device helpers for libmcb200 (sm_100a only).
// Nothing in this tree is shared with oracle/ (the CPU checker).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mcb {

constexpr int kTile = 32;            // chain tile: one warp lane per particle
constexpr int kChunkMax = 1024;      // rows resolved by one chain kernel (max)
constexpr int kColTile = 128;        // columns staged per bulk-copy stage
constexpr int kStages = 4;           // smem ring depth of the bulk kernel
constexpr int kBulkThreads = 256;    // consumer threads per bulk CTA (each owns 1 or 2 rows)
constexpr int kMaxSlices = 512;      // upper bound on column slices of the bulk kernel
constexpr double kGhostCoord = 1.0e9;
constexpr double kGhostStep = 1.0e6;

// flags of the trial log (same meaning as in include/mcb200.h)
constexpr unsigned kFlagAccept = 1u, kFlagOverlap = 2u, kFlagWall = 4u, kFlagNearTie = 8u;

struct DevState {
    unsigned long long sweep;
    unsigned long long accepted, veto_overlap, veto_wall, near_ties;
    double E_run;
    int err;        // validation result (0 ok, MC_E* otherwise)
    int d_differs;  // set by k_check_particles if not all diameters are equal
    int stall;      // set by the sweep kernel's watchdog (a wait exceeded its time limit)
    int sched_mismatch;   // sweeps whose per-chunk completion counters did not equal the plan's item counts (must stay 0)
    unsigned long long dmin_bits;   // bit pattern of the smallest diameter (k_check_particles; ~0 before)
};

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), written from the round description; reading G9.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// u = (2k+1) 2^-53, k = top 52 bits of (hi:lo); exact, in (0,1).  Reading G10.
__device__ __forceinline__ double uniform_open01(uint32_t lo, uint32_t hi) {
    const unsigned long long w = ((unsigned long long)hi << 32) | lo;
    const unsigned long long k = w >> 12;
    return __ull2double_rn(2ull * k + 1ull) * 0x1.0p-53;
}

// r^2 in the evaluation order fixed by reading G11: fma(dz,dz,fma(dy,dy,dx*dx)).
__device__ __forceinline__ double dist2(double dx, double dy, double dz) {
    return __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
}

// 1/sqrt(x) for normal positive x: MUFU.RSQ64H seed + one cubic refinement
// (e = 1 - x y^2;  y <- y (1 + e (1/2 + 3/8 e))), 5 FP64-pipe instructions, no slow path, within 2 ulp.
// Written so that NO instruction reads three different registers: on B200 a DFMA with three distinct register
// operands occupies the FP64 pipe for 3 cycles instead of 2 (measured: 66 % of the DMUL / DADD rate; with an
// immediate or a repeated operand 98 %).  The usual last step y + (y e) p is such an
// instruction; y (1 + e p) is not.
__device__ __forceinline__ double rsqrt_fast(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = __dmul_rn(x, y);
    const double e = __fma_rn(-t, y, 1.0);
    const double p = __fma_rn(0.375, e, 0.5);
    const double q = __fma_rn(e, p, 1.0);
    return __dmul_rn(y, q);
}

// ---------------------------------------------------------------------------------------------
// mbarrier + 1-D bulk async copy (cp.async.bulk; SASS UBLKCP) wrappers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(
                     smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
// global -> shared bulk copy; bytes multiple of 16, both addresses 16-byte aligned.
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes,
                                         uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(smem_dst)),
        "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace mcb
