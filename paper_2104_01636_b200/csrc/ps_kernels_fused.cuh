// ps_kernels_fused.cuh -- fused red+black z-marching sweep kernels (sm_100a).  [stub: first slice]
#pragma once
#include <cuda_runtime.h>

#include "ps_kernels_generic.cuh"

namespace ps {

struct FusedPlan {
    int sm_count;
};

inline bool fused_shape_ok(const Grid &) { return false; }

inline cudaError_t fused_plan_init(FusedPlan *pl, const Grid &, int sm_count)
{
    pl->sm_count = sm_count;
    return cudaSuccess;
}

inline cudaError_t launch_fused(const FusedPlan &, const Grid &, const double *, const double *,
                                const double *, const double *, const double *, double *, double,
                                int, cudaStream_t, int *did)
{
    *did = 0;
    return cudaErrorNotSupported;
}

}  // namespace ps
