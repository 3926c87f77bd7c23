// cos_kernels_typed.cuh -- instantiates the precision-generic kernels twice:
//   cosb::f64  real = double   the product path (north_star: FP64 everywhere)
//   cosb::f32  real = float    the FP32 variant of SURVEY.md 8(f2) (the paper's own operating point)
#pragma once
#include "cos_common.cuh"
#include "cos_kernels_generic.cuh"

namespace cosb {

__device__ __forceinline__ float sel(bool p, float a, float b) { return p ? a : b; }
__device__ __forceinline__ void leaf_conv(const float (&c)[16], const float (&dd)[16], float (&acc)[16])
{
#pragma unroll
    for (int S = 0; S < 16; ++S)
#pragma unroll
        for (int T = 0; T < 16; ++T)
            if ((T & ~S) == 0) acc[S] = fmaf(c[T], dd[S ^ T], acc[S]);
}

namespace f64 {
using real = double;
using real2 = double2;
__device__ __forceinline__ real2 make_real2(real a, real b) { return make_double2(a, b); }
__device__ __forceinline__ const real* in_real(const double* p) { return p; }
#include "cos_eval_generic.inc"
#include "cos_eval_team.inc"
#include "cos_eval_pair.inc"
}  // namespace f64

namespace f32 {
using real = float;
using real2 = float2;
__device__ __forceinline__ real2 make_real2(real a, real b) { return make_float2(a, b); }
__device__ __forceinline__ const real* in_real(const double* p) { return reinterpret_cast<const real*>(p); }
#include "cos_eval_generic.inc"
#include "cos_eval_team.inc"
#include "cos_eval_pair.inc"
}  // namespace f32

}  // namespace cosb
