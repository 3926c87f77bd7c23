// cos_mc.cuh -- on-device Monte Carlo over the vertex coordinates (reading R19).
//
// P:47 "The integration over the vertex coordinates can then be performed by stochastic (Monte Carlo) sampling";
// P:137 "one needs to handle proposal and acceptance of configurations ... readily implemented in device-sided
// code"; "many Markov chain walkers ... localised to a single GPU".  The paper gives no update scheme; reading
// R19 fixes the plainest one.  One walker = one configuration of the batch, weight |connected(x)|, one update per
// step (vertex k = r0 mod n re-drawn uniformly in space and time, a symmetric proposal), accepted iff
// u * |w_old| < |w_new|.  Random numbers come from philox4x32-10 (Salmon et al., SC'11), a counter-based generator
// keyed by the seed and addressed by (step, stream, walker): no generator state lives in memory, any thread can
// recompute the draws of its walker, and the sequence does not depend on the launch shape.
// The evaluation of the proposals is the ordinary hot path (cos_build_G + evaluation kernel over the whole batch of
// walkers); the two kernels here only move coordinates.
#pragma once
#include "cos_common.cuh"

namespace cosb {

struct Philox4 { uint32_t v[4]; };

__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    Philox4 r;
    r.v[0] = c0; r.v[1] = c1; r.v[2] = c2; r.v[3] = c3;
    return r;
}

// 53 random bits -> [0, 1)
__device__ __forceinline__ double u53(uint32_t a, uint32_t b)
{
    const unsigned long long x = ((unsigned long long)a << 21) ^ ((unsigned long long)b >> 11);
    return (double)x * (1.0 / 9007199254740992.0);
}

struct McArgs {
    int n;
    long long walkers;
    int step;
    unsigned long long seed;
    int Lx, Ly;
    double beta;
    int* xy;                 // [walkers][n][2] state
    double* tau;             // [walkers][n]
    int* xy_p;               // proposal
    double* tau_p;
    const double* w_old;     // [walkers] weight of the state before this step
    const double* w_new;     // [walkers] weight of the proposal
    double* w_out;           // [walkers] weight of the state after this step
    unsigned char* hist;     // nullptr or [steps][walkers]
    long long* accepted;     // nullptr or [walkers]
    double* sign_sum;        // nullptr or [walkers]
};

// One thread per (walker, vertex): the proposal is the state with vertex k of the walker re-drawn.
__global__ void __launch_bounds__(256) mc_propose_kernel(McArgs a)
{
    const long long total = a.walkers * a.n;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long w = t / a.n;
        const int v = (int)(t - w * a.n);
        const uint32_t k0 = (uint32_t)a.seed, k1 = (uint32_t)(a.seed >> 32);
        const Philox4 r = philox4x32_10((uint32_t)a.step, 0u, (uint32_t)w, (uint32_t)((unsigned long long)w >> 32), k0, k1);
        const int k = (int)(r.v[0] % (uint32_t)a.n);
        int x = a.xy[2 * t], y = a.xy[2 * t + 1];
        double tv = a.tau[t];
        if (v == k) {
            const Philox4 s = philox4x32_10((uint32_t)a.step, 1u, (uint32_t)w, (uint32_t)((unsigned long long)w >> 32), k0, k1);
            x = (int)(r.v[1] % (uint32_t)a.Lx);
            y = (int)(r.v[2] % (uint32_t)a.Ly);
            tv = a.beta * u53(s.v[0], s.v[1]);
        }
        a.xy_p[2 * t] = x;
        a.xy_p[2 * t + 1] = y;
        a.tau_p[t] = tv;
    }
}

// One thread per (walker, vertex): Metropolis decision of the walker, then the accepted proposal replaces the state.
__global__ void __launch_bounds__(256) mc_accept_kernel(McArgs a)
{
    const long long total = a.walkers * a.n;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long w = t / a.n;
        const int v = (int)(t - w * a.n);
        const uint32_t k0 = (uint32_t)a.seed, k1 = (uint32_t)(a.seed >> 32);
        const Philox4 s = philox4x32_10((uint32_t)a.step, 1u, (uint32_t)w, (uint32_t)((unsigned long long)w >> 32), k0, k1);
        const double wo = a.w_old[w], wn = a.w_new[w];
        const bool ok = u53(s.v[2], s.v[3]) * fabs(wo) < fabs(wn);      // symmetric proposal: min(1, |w_new| / |w_old|)
        if (ok) {
            a.xy[2 * t] = a.xy_p[2 * t];
            a.xy[2 * t + 1] = a.xy_p[2 * t + 1];
            a.tau[t] = a.tau_p[t];
        }
        if (v == 0) {
            const double wc = ok ? wn : wo;
            a.w_out[w] = wc;
            if (a.hist) a.hist[(long long)a.step * a.walkers + w] = ok ? 1 : 0;
            if (a.accepted && ok) a.accepted[w] += 1;
            if (a.sign_sum) a.sign_sum[w] += (double)((wc > 0.0) - (wc < 0.0));
        }
    }
}

}  // namespace cosb
