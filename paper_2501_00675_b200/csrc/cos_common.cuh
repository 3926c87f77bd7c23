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
    const uint32_t* off;   // off[R] = sum_{x<R}(popc(x)+1), R = 0..2^(kMaxN-1)
    double* scratch;       // per-CTA global scratch (large n), may be nullptr
    size_t scratch_stride; // doubles per CTA
    int fused;             // unused (no kernel assembles G on the fly any more); kept 0
    const unsigned char* tabs;   // team kernel: table image of this order built once per context (or nullptr)
    BuildGArgs bg;
};

}  // namespace cosb
