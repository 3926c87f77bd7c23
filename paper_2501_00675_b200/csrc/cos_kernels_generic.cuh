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
// One thread per entry (i, j) of a configuration; a CTA stages the vertices of kBuildGCfgs configurations in shared
// memory (coalesced loads) and walks the batch grid-strided.  Table rows are L2 resident (1-8 MiB); two adjacent
// tau points per entry.

// x / beta, correctly rounded, with the reciprocal y = RN(1 / beta) taken once on the host (Markstein's sequence for a
// loop-invariant divisor: two FMA refinements, the residuals are exact and the last FMA rounds the quotient like a
// division does).  The result is bit-identical to __ddiv_rn(x, beta); outside the range where the residuals cannot
// underflow or overflow -- and when the host found the all-ones significand the theorem excludes -- the division
// itself is used.  The kernel spent half of its instructions in the generic division.
__device__ __forceinline__ double div_by_beta(const BuildGArgs& a, double x)
{
    if (!a.fast_div || !(x > 1e-200 && x < 1e200)) return __ddiv_rn(x, a.beta);
    const double y = a.rbeta, b = a.beta;
    double q = __dmul_rn(x, y);
    double r = __fma_rn(-b, q, x);
    q = __fma_rn(r, y, q);
    r = __fma_rn(-b, q, x);
    return __fma_rn(r, y, q);
}

// Off-diagonal value from the coordinates of the two vertices (reading R8: 2-point lerp on the tau grid,
// antiperiodic branch for dtau <= 0, R9).
__device__ __forceinline__ void g0_value(const BuildGArgs& a, int xi, int yi, int xj, int yj, double ti, double tj,
                                         double& gup, double& gdn)
{
    // sites arrive reduced to [0, L) (build_G_kernel reduces them once per vertex when it stages them), so the
    // difference needs one conditional add instead of a division
    int dx = xi - xj, dy = yi - yj;
    if (dx < 0) dx += a.Lx;
    if (dy < 0) dy += a.Ly;
    double dtau = ti - tj;
    double sign = 1.0;
    if (dtau <= 0.0) { dtau = __dadd_rn(dtau, a.beta); sign = -1.0; }     // R9: dtau == 0 is 0-
    const double uu = div_by_beta(a, __dmul_rn(dtau, (double)(a.ntau - 1)));
    int k = (uu >= 2147483647.0) ? a.ntau - 2 : __double2int_rd(uu);      // floor; NaN and negatives clamp to 0 below
    k = min(k, a.ntau - 2);
    k = max(k, 0);
    const double f = __dsub_rn(uu, (double)k);
    const unsigned row = (unsigned)(dx * a.Ly + dy) * (unsigned)a.ntau + (unsigned)k;     // tables are < 2^32 entries (cos_set_g0_table)
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

constexpr int kBuildGThreads = 256;    // at most: the launch uses build_G_threads(n)
constexpr int kBuildGCfgs = 8;         // configurations staged per CTA pass (measured at n = 10, batch 16384: 4: 25.5, 8: 23.1, 16: 24.9 us)
// Threads per CTA: as many whole configurations as fit in 256 threads, one thread per entry, rounded up to a warp.
__host__ __device__ inline int build_G_threads(int n) { return ((kBuildGThreads / (n * n)) * (n * n) + 31) & ~31; }

__global__ void __launch_bounds__(kBuildGThreads) build_G_kernel(BuildGArgs a)
{
    __shared__ int sx[kBuildGCfgs * kMaxN], sy[kBuildGCfgs * kMaxN];
    __shared__ double st[kBuildGCfgs * kMaxN];
    const int n = a.n, nn = n * n;
    // a thread keeps its entry (i, j) for the whole launch and walks the configurations of a pass in steps of
    // per_pass: every index inside the loop advances by a constant
    const int per_pass = kBuildGThreads / nn;
    const int cl = (int)threadIdx.x / nn, e = (int)threadIdx.x - cl * nn, i = e / n, j = e - i * n;
    const bool live = cl < per_pass;
    for (long long b0 = (long long)blockIdx.x * kBuildGCfgs; b0 < a.batch; b0 += (long long)gridDim.x * kBuildGCfgs) {
        const int cfgs = (int)min((long long)kBuildGCfgs, a.batch - b0);
        const int* xy = a.xy + b0 * n * 2;
        const double* tau = a.tau + b0 * n;
        __syncthreads();                                   // the previous pass has read its vertices
        for (int v = threadIdx.x; v < cfgs * n; v += blockDim.x) {
            int x = xy[2 * v], y = xy[2 * v + 1];
            if ((unsigned)x >= (unsigned)a.Lx) { x %= a.Lx; if (x < 0) x += a.Lx; }      // (x_i - x_j) mod L from the residues
            if ((unsigned)y >= (unsigned)a.Ly) { y %= a.Ly; if (y < 0) y += a.Ly; }
            sx[v] = x; sy[v] = y; st[v] = tau[v];
        }
        __syncthreads();
        if (!live) continue;
        double* gu = a.Gup + b0 * nn + e;
        double* gd = a.Gdn ? a.Gdn + b0 * nn + e : nullptr;
        for (int c = cl; c < cfgs; c += per_pass) {        // consecutive threads: consecutive entries
            const int vi = c * n + i, vj = c * n + j;
            double gup = a.g_diag, gdn = a.g_diag;
            if (i != j) g0_value(a, sx[vi], sy[vi], sx[vj], sy[vj], st[vi], st[vj], gup, gdn);
            gu[c * nn] = gup;
            if (gd) gd[c * nn] = gdn;
        }
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
