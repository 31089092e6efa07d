// rt_slab.cuh -- large-batch variant of fused steps 1-4 (placeholder until the staged kernel lands)
#pragma once
#include "common.cuh"

namespace helios {

struct SlabArgs {
    const float* sigma; const float* cia;
    int S, C, nT, nP, nNu, L, B;
    long long stride;
    const int* lvl_ip; const float* lvl_u;
    const float* rec; int rec_floats;
    const float* model_scale; const int* model_flag;
    double nu0, dnu;
    float* flux; long long flux_stride;
    AngleSet ang;
};

inline bool slab_supported(int, int, int, int) { return false; }
inline cudaError_t launch_rt_slab(const SlabArgs&, int, int, int, cudaStream_t, int*) { return cudaErrorNotSupported; }

}  // namespace helios
