// sweep_inst.cu -- the k_sweep instantiations of one pair-distance form (MCB_FORM = 0 GRAM, 1 DIFFW, 2 CANON).
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false -DMCB_FORM=<f> -c
#include "sweep_launch.h"

#ifndef MCB_FORM
#error "compile with -DMCB_FORM=0|1|2"
#endif

#define MCB_CAT2(a, b) a##b
#define MCB_CAT(a, b) MCB_CAT2(a, b)
#define MCB_FORM_NS MCB_CAT(form, MCB_FORM)

namespace mcb {
namespace MCB_FORM_NS {

template <int ROWS, bool UNIFORM>
static int launch_one(const SweepLaunch& L, int* ctas_per_sm) {
    auto kern = k_sweep<ROWS, UNIFORM, MCB_FORM>;
    const int smem = (int)sizeof(PShared);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return (int)e;
    if (L.grid == 0) {
        return (int)cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, kern, kPThreads, smem);
    }
    PArgs a = L.args;
    void* args[] = {(void*)&a};
    return (int)cudaLaunchCooperativeKernel((void*)kern, dim3(L.grid), dim3(kPThreads), args, (size_t)smem, L.stream);
}

static int launch_any(const SweepLaunch& L, int* ctas_per_sm) {
    switch (L.rows) {
        case 1: return L.uniform ? launch_one<1, true>(L, ctas_per_sm) : launch_one<1, false>(L, ctas_per_sm);
        case 2: return L.uniform ? launch_one<2, true>(L, ctas_per_sm) : launch_one<2, false>(L, ctas_per_sm);
        case 3: return L.uniform ? launch_one<3, true>(L, ctas_per_sm) : launch_one<3, false>(L, ctas_per_sm);
        default: return L.uniform ? launch_one<4, true>(L, ctas_per_sm) : launch_one<4, false>(L, ctas_per_sm);
    }
}

}  // namespace MCB_FORM_NS

#if MCB_FORM == 0
int launch_sweep_gram(const SweepLaunch& L, int* c) { return MCB_FORM_NS::launch_any(L, c); }
#elif MCB_FORM == 1
int launch_sweep_diffw(const SweepLaunch& L, int* c) { return MCB_FORM_NS::launch_any(L, c); }
#else
int launch_sweep_canon(const SweepLaunch& L, int* c) { return MCB_FORM_NS::launch_any(L, c); }
#endif

}  // namespace mcb
