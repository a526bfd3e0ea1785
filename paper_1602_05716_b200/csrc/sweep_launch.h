// sweep_launch.h -- how mcb200.cu reaches the instantiations of k_sweep, which are compiled one pair-distance
// form per translation unit (sweep_inst.cu with -DMCB_FORM=0|1|2) so that the library builds in parallel.
#pragma once
#include "persist.cuh"

namespace mcb {

struct SweepLaunch {
    PArgs args;
    int rows;          // rows per consumer thread: 1 to 4
    bool uniform;      // all diameters equal
    int grid;          // CTAs (0: query only)
    cudaStream_t stream;
};

// Returns a cudaError_t.  With grid == 0 only *ctas_per_sm is filled (occupancy of the instantiation,
// after raising its dynamic shared memory limit); otherwise launches cooperatively.
int launch_sweep_gram(const SweepLaunch& L, int* ctas_per_sm);
int launch_sweep_diffw(const SweepLaunch& L, int* ctas_per_sm);
int launch_sweep_canon(const SweepLaunch& L, int* ctas_per_sm);

}  // namespace mcb
