// hydro_stage_fused.cuh -- placeholder until the tiled fused stage kernel lands (next commit).
#pragma once
#include "hydro_kernels.cuh"

namespace hyd {

struct FusedPlan { int ready = 0; };

inline cudaError_t plan_stage_fused(FusedPlan &, const Grid &, const double *, const double *)
{
    return cudaSuccess;
}

template <int STAGE>
inline cudaError_t launch_stage_fused(const FusedPlan &, const Grid &, const double *, const double *,
                                      double *, double, const StepScalars *, double, StepScalars *,
                                      cudaStream_t)
{
    return cudaErrorNotSupported;
}

}  // namespace hyd
