// cos_kernels_generic.cuh -- generic (any n in 1..16) CoS evaluation kernel and the G-assembly kernel.
//
// This is the reference-correct CUDA path: one CTA per configuration, grid-strided over the batch,
// the whole path a2..a5 inside one kernel.  It is the fallback for orders that have no specialised
// kernel and the kernel every specialised variant is tested against (besides the oracle).
//
// Method (reading R1):
//   nodes (S, c): S = vertex subset, c in S = current end of the open path that started at h(S) = max S.
//   Organised by "stage" h = h(S): stage h works on R = S \ {h}, R subset of [h] = {0..h-1}:
//       P_h[R][h]  = Z[R]                                            (start a loop at h)
//       P_h[R+c'][c'] = sum_{c in R+{h}} P_h[R][c] * W[c][c']  c' not in R   (extend)
//       Z[R+{h}]   = - sum_{c in R+{h}} P_h[R][c] * W[c][h]          (close, -1 per fermion loop)
//   levels j = |R| = 0..h are processed in sequence with a block barrier, stages in sequence
//   because stage h reads every Z[R], R subset of [h].  Z[S] = (-1)^|S| det W[S,S] for every S.
//   Then D[S] = w(S) Zup[S] Zdn[S] and the subset recursion for the connected part.
#pragma once
#include "cos_common.cuh"

namespace cosb {

// ------------------------------------------------------------------------------------------ a1
// One thread per (b, i, j).  Table rows are L2 resident (1-8 MiB); two adjacent tau points per entry.
// One entry G_s[b][i][j] (both species) of step a1.
// Off-diagonal value from the coordinates of the two vertices (reading R8: 2-point lerp on the tau grid,
// antiperiodic branch for dtau <= 0, R9).
__device__ __forceinline__ void g0_value(const BuildGArgs& a, int xi, int yi, int xj, int yj, double ti, double tj,
                                         double& gup, double& gdn)
{
    int dx = (xi - xj) % a.Lx; if (dx < 0) dx += a.Lx;
    int dy = (yi - yj) % a.Ly; if (dy < 0) dy += a.Ly;
    double dtau = ti - tj;
    double sign = 1.0;
    if (dtau <= 0.0) { dtau = __dadd_rn(dtau, a.beta); sign = -1.0; }     // R9: dtau == 0 is 0-
    const double uu = __ddiv_rn(__dmul_rn(dtau, (double)(a.ntau - 1)), a.beta);
    int k = (int)floor(uu);
    k = min(k, a.ntau - 2);
    k = max(k, 0);
    const double f = __dsub_rn(uu, (double)k);
    const size_t row = ((size_t)dx * a.Ly + dy) * (size_t)a.ntau + k;
    {
        const double t0 = __ldg(a.Tup + row), t1 = __ldg(a.Tup + row + 1);
        gup = sign * __fma_rn(f, __dsub_rn(t1, t0), t0);
    }
    if (a.Tdn && a.Tdn != a.Tup) {
        const double t0 = __ldg(a.Tdn + row), t1 = __ldg(a.Tdn + row + 1);
        gdn = sign * __fma_rn(f, __dsub_rn(t1, t0), t0);
    } else {
        gdn = gup;
    }
}

__device__ __forceinline__ void g0_entry(const BuildGArgs& a, long long b, int i, int j, double& gup, double& gdn)
{
    if (i == j) { gup = a.g_diag; gdn = a.g_diag; return; }
    const int* pi = a.xy + (b * a.n + i) * 2;
    const int* pj = a.xy + (b * a.n + j) * 2;
    g0_value(a, pi[0], pi[1], pj[0], pj[1], a.tau[b * a.n + i], a.tau[b * a.n + j], gup, gdn);
}

// One thread per (b, i, j); a CTA walks whole configurations so that the index arithmetic stays 32-bit.
__global__ void __launch_bounds__(256) build_G_kernel(BuildGArgs a)
{
    const int nn = a.n * a.n;
    const int per_cta = 256 / nn > 0 ? 256 / nn : 1;          // configurations per CTA pass (n <= 16: nn <= 256)
    const int local = threadIdx.x / nn, e = threadIdx.x - local * nn;
    if (local >= per_cta) return;
    const int i = e / a.n, j = e - i * a.n;
    for (long long b = (long long)blockIdx.x * per_cta + local; b < a.batch; b += (long long)gridDim.x * per_cta) {
        double gup, gdn;
        g0_entry(a, b, i, j, gup, gdn);
        a.Gup[b * nn + e] = gup;
        if (a.Gdn) a.Gdn[b * nn + e] = gdn;
    }
}

// off[R] = sum_{x<R} (popc(x)+1): slot of node (R, first element) when the nodes of one stage are
// stored in numeric order of R, each R holding popc(R)+1 values (elements of R ascending, then h).
__global__ void init_off_table_kernel(uint32_t* off, uint32_t count)
{
    // single block, serial prefix per thread chunk is unnecessary: count <= 32769, do a simple scan.
    __shared__ uint32_t partial[1024];
    const uint32_t per = (count + blockDim.x - 1) / blockDim.x;
    const uint32_t lo = threadIdx.x * per, hi = min(count, lo + per);
    uint32_t s = 0;
    for (uint32_t x = lo; x < hi; ++x) s += __popc(x) + 1;
    partial[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0;
        for (unsigned t = 0; t < blockDim.x; ++t) { const uint32_t v = partial[t]; partial[t] = run; run += v; }
    }
    __syncthreads();
    s = partial[threadIdx.x];
    for (uint32_t x = lo; x < hi; ++x) { off[x] = s; s += __popc(x) + 1; }
}

// Shared-memory footprint of the generic kernel, in doubles.
//   W: 2*n*n, u: n (padded to 16), Z: nsp * 2^n, P: (n+1) 2^(n-2) (stage n-1; also holds C' later)
__host__ __device__ inline size_t generic_frontier_doubles(int n)
{
    return n >= 2 ? ((size_t)(n + 1) << (n - 2)) : 2;
}
__host__ __device__ inline size_t generic_small_doubles(int n) { return (size_t)2 * n * n + 16; }

}  // namespace cosb
