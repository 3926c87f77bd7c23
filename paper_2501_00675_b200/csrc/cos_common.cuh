// cos_common.cuh -- shared declarations of the CUDA path (sm_100a).  No oracle code is included here.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/cos.h"

namespace cosb {

constexpr int kMaxN = COS_MAX_ORDER;

// Arguments of the G-assembly launch (step a1).
struct BuildGArgs {
    int n;
    long long batch;
    const int* xy;        // [batch][n][2]
    const double* tau;    // [batch][n]
    const double* Tup;    // [Lx][Ly][ntau]
    const double* Tdn;    // == Tup when shared
    int Lx, Ly, ntau;
    double beta;
    double rbeta;         // RN(1 / beta), taken on the host
    int fast_div;         // 1: x / beta by the FMA sequence of div_by_beta (0: the significand of beta is all ones)
    double g_diag;
    double* Gup;          // [batch][n][n]
    double* Gdn;          // nullptr: write Gup only
};

// Arguments of one evaluation launch (steps a2..a5 of SURVEY.md §8(a)).
struct EvalArgs {
    int n;
    long long batch;
    const double* Gup;     // [batch][n][n]
    const double* Gdn;     // [batch][n][n]; == Gup when the species share one matrix
    const double* u;       // [batch][n] or nullptr
    double U;
    double* out;           // [batch]
    int connected;         // 0: D[full] ("all"), 1: C[full]
    int halfvertex;        // 1: half-vertex formulation (reading R18): n = 2n' points, one species, u = V [batch][n'];
                           //    generic kernel only
    double loopf;          // factor of one closed fermion loop: -1, or -N_f (cos_set_loop_weight, reading R17)
    const uint32_t* off;   // off[R] = sum_{x<R}(popc(x)+1), R = 0..2^(kMaxN-1)
    double* scratch;       // per-CTA global scratch (large n), may be nullptr
    size_t scratch_stride; // doubles per CTA
    const unsigned char* tabs;   // team kernel: table image of this order built once per context (or nullptr)
};

// Binomial coefficients (subset ranks in colex order), device and host copies.
struct Binom {
    int c[18][18];
};
constexpr Binom make_binom()
{
    Binom b{};
    for (int i = 0; i < 18; ++i) {
        b.c[i][0] = 1;
        for (int j = 1; j < 18; ++j) b.c[i][j] = (i == 0) ? 0 : b.c[i - 1][j - 1] + b.c[i - 1][j];
    }
    return b;
}
__constant__ Binom kBinom = make_binom();
constexpr Binom kBinomHost = make_binom();

__host__ __device__ constexpr int cpopc(int x) { int c = 0; while (x) { c += x & 1; x >>= 1; } return c; }

__device__ __forceinline__ double sel(bool p, double a, double b) { return p ? a : b; }

// Subset convolution of two blocks over the 4 lowest vertices: acc[S] += sum_{T subset of S} c[T] * dd[S \ T]
// (81 FMAs on 32 values; the leaf of the connected reduction).
__device__ __forceinline__ void leaf_conv(const double (&c)[16], const double (&dd)[16], double (&acc)[16])
{
#pragma unroll
    for (int S = 0; S < 16; ++S)
#pragma unroll
        for (int T = 0; T < 16; ++T)
            if ((T & ~S) == 0) acc[S] = fma(c[T], dd[S ^ T], acc[S]);
}

#ifdef COS_PHASE_TIMING
// Development aid (-DCOS_PHASE_TIMING builds only): cycles thread 0 of every CTA spent per phase, summed over CTAs.
__device__ unsigned long long g_phase_cycles[32];
#define COS_PHASE_MARK(k) do { __syncthreads(); if (threadIdx.x == 0) { const long long now__ = clock64(); \
    atomicAdd(&g_phase_cycles[k], (unsigned long long)(now__ - phase_t0__)); phase_t0__ = now__; } } while (0)
#else
#define COS_PHASE_MARK(k) do { } while (0)
#endif

}  // namespace cosb
