// cos_dispatch.cuh -- picks the kernel variant for an evaluation launch and sizes its resources.
#pragma once
#include "cos_common.cuh"
#include "cos_kernels_generic.cuh"
#include "cos_kernels_tiled.cuh"
#include "cos_kernels_team.cuh"
#include "cos_kernels_pair.cuh"

namespace cosb {

constexpr int kGenericThreads = 256;
constexpr int kTiledB = 3;
constexpr int kTiledThreads = 128;
constexpr int kTiledNA = 4, kTiledJB = 5;
constexpr int kTiledMinN = 5, kTiledMaxN = 12;

inline size_t generic_smem_bytes(int n, int nsp)
{
    return sizeof(double) * (generic_small_doubles(n) + ((size_t)nsp << n) + generic_frontier_doubles(n));
}

// True when the generic kernel must keep Z and the frontier in global scratch.
inline bool generic_needs_global(int n, int smem_optin)
{
    return generic_smem_bytes(n, 2) > (size_t)smem_optin;
}

// Configurations per CTA of the tiled kernel (0: the tiled kernel cannot run this order).
inline int tiled_group(int n, int nsp, int smem_optin)
{
    if (n < kTiledMinN || n > kTiledMaxN) return 0;
    if (tiled_smem_bytes<kTiledB>(n, 1, nsp) > (size_t)smem_optin) return 0;
    const int q = n - kTiledB - 1;                       // widest stage
    const int widest = kBinomHost.c[q][q / 2];
    int G = (kTiledThreads + widest - 1) / widest;
    const size_t budget = 112 * 1024;                    // keep two CTAs per SM where possible
    while (G > 1 && tiled_smem_bytes<kTiledB>(n, G, nsp) > budget) --G;
    return G;
}

inline bool uses_tiled(int n, int nsp, int smem_optin) { return tiled_group(n, nsp, smem_optin) > 0; }

// Orders 13..16: the tiled kernel with one configuration per CTA whose block (W, Z, level buffers, reduction
// arrays) lives in global scratch (L2 resident); only the subset tables stay in shared memory.
constexpr int kBigThreads = 256, kBigNA = 6, kBigJB = 7, kBigMinN = 13;
inline bool uses_big(int n) { return n >= kBigMinN && n <= kMaxN; }
inline TiledDims big_dims(int n, int nsp)
{
    TiledDims d = tiled_dims<kTiledB>(n, 1, nsp);
    d.use_global = 1;
    return d;
}

inline size_t pair_global_rec_doubles(int n);   // defined with the pair-kernel choices below

// Doubles of global scratch per CTA (0: everything lives in shared memory).
inline size_t eval_scratch_doubles(int n, int smem_optin)
{
    if (uses_big(n)) {
        size_t v = (size_t)big_dims(n, 2).cfg_doubles;
        const size_t p = pair_global_rec_doubles(n);     // the pair kernel on global records (orders 14..16)
        if (p > v) v = p;
        return v;
    }
    if (uses_tiled(n, 2, smem_optin)) return 0;
    if (!generic_needs_global(n, smem_optin)) return 0;
    return ((size_t)2 << n) + generic_frontier_doubles(n);
}

inline int eval_max_ctas(int n, long long batch, int num_sms, int smem_optin)
{
    (void)n; (void)smem_optin;
    const long long cap = (long long)num_sms * 2;
    return (int)(batch < cap ? batch : cap);
}

// ---- team kernel (orders 5..10): instances per team and launch shape per order ----
constexpr int kTeamMinN = 5, kTeamMaxN = 10;
using TeamKernel = void (*)(EvalArgs, TeamDims);
struct TeamChoice { TeamKernel fn; TeamDims d; };
inline bool uses_team(int n) { return n >= kTeamMinN && n <= kTeamMaxN; }
inline TeamChoice team_choice(int n, int nsp)
{
    if (n == 10) return {eval_team_kernel<4, 160, 2>, team_dims<4>(n, nsp)};
    if (n == 9) return {eval_team_kernel<8, 160, 2>, team_dims<8>(n, nsp)};
    if (n == 8) return {eval_team_kernel<16, 160, 2>, team_dims<16>(n, nsp)};
    return {eval_team_kernel<32, 192, 2>, team_dims<32>(n, nsp)};
}

// ---- pair kernel (orders 11..12): the team mapping with every item split over a lane pair ----
constexpr int kPairMinN = 11, kPairMaxN = 13;
using PairKernel = void (*)(EvalArgs, PairDims);
struct PairChoice { PairKernel fn; PairDims d; };
inline bool uses_pair(int n) { return n >= kPairMinN && n <= kPairMaxN; }
// True when order n has a kernel that assembles G on the fly (cos_eval_connected_xt without a G round trip).
inline bool has_fused_kernel(int n, int nsp, int smem_optin);
inline PairChoice pair_choice(int n, int nsp)
{
    if (n == 13) return {eval_pair_kernel<1, 512, 1, 10>, pair_dims<1>(n, 1)};   // one species only (see dispatch_eval)
    if (n == 12) return {eval_pair_kernel<2, 512, 1, 9>, pair_dims<2>(n, nsp)};
    return {eval_pair_kernel<4, 512, 1, 8>, pair_dims<4>(n, nsp, 512)};
}

// No evaluation kernel assembles G on the fly any more: a separate cos_build_G launch plus a cp.async prefetch of
// the next team's matrices measured faster than the in-kernel gather (whose two dependent global round trips per
// team sat on the critical path), and G costs 16 n^2 bytes per configuration of HBM traffic -- noise.
inline bool has_fused_kernel(int, int, int) { return false; }

// ---- pair kernel on global records (orders 14..16, one species): Z / frontier / reduction arrays in L2 scratch ----
constexpr int kPairGlobalMinN = 14, kPairGlobalThreads = 512;
// one species: C = 1 from order 14; two species (G_up != G_down): C = 2 (the two instances of one configuration)
// from order 13, where the shared-memory variant has room for one instance only
inline bool uses_pair_global(int n, int nsp)
{
    return n <= kMaxN && (nsp == 1 ? n >= kPairGlobalMinN : n >= kPairGlobalMinN - 1);
}
inline PairChoice pair_global_choice(int n, int nsp = 1)
{
    if (nsp == 2) return {eval_pair_kernel<2, kPairGlobalThreads, 1, 8, true>, pair_dims_global<2>(n, kPairGlobalThreads, 2)};
    return {eval_pair_kernel<1, kPairGlobalThreads, 1, 8, true>, pair_dims_global<1>(n, kPairGlobalThreads)};
}
inline size_t pair_global_rec_doubles(int n)
{
    if (n < kPairGlobalMinN - 1 || n > kMaxN) return 0;
    const size_t a = (size_t)pair_global_choice(n, 1).d.rec_doubles, b = (size_t)pair_global_choice(n, 2).d.rec_doubles;
    return a > b ? a : b;
}

using TiledKernel = void (*)(EvalArgs, TiledDims);
inline TiledKernel tiled_kernel() { return eval_tiled_kernel<kTiledB, kTiledThreads, kTiledNA, kTiledJB, false>; }
inline TiledKernel big_kernel() { return eval_tiled_kernel<kTiledB, kBigThreads, kBigNA, kBigJB, true>; }

inline cudaError_t configure_kernels(int smem_optin)
{
    cudaError_t e = cudaFuncSetAttribute(eval_generic_kernel<kGenericThreads>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
    for (int n = kTeamMinN; n <= kTeamMaxN; ++n) {
        e = cudaFuncSetAttribute(team_choice(n, 1).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (e != cudaSuccess) return e;
    }
    for (int n = kPairMinN; n <= kPairMaxN; ++n) {
        e = cudaFuncSetAttribute(pair_choice(n, 1).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (e != cudaSuccess) return e;
    }
    e = cudaFuncSetAttribute(pair_global_choice(kPairGlobalMinN, 1).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(pair_global_choice(kPairGlobalMinN, 2).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(big_kernel(), cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(tiled_kernel(), cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
}

inline cudaError_t dispatch_eval(const EvalArgs& a, cudaStream_t stream, int num_sms, int smem_optin,
                                 int* launches, const char** name)
{
    const int nsp = a.fused ? (a.bg.Tdn != a.bg.Tup ? 2 : 1) : ((a.Gdn == a.Gup) ? 1 : 2);
    *launches = 1;
    if (uses_team(a.n)) {
        const TeamChoice tc = team_choice(a.n, nsp);
        if (tc.d.smem_bytes <= (size_t)smem_optin) {
            int per_sm = 1;
            const int block = tc.d.threads;
            cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tc.fn, block, tc.d.smem_bytes);
            if (e != cudaSuccess) return e;
            if (per_sm < 1) per_sm = 1;
            const long long teams = (a.batch * nsp + tc.d.C - 1) / tc.d.C;
            long long grid = (long long)num_sms * per_sm;
            if (grid > teams) grid = teams;
            tc.fn<<<(unsigned)grid, block, tc.d.smem_bytes, stream>>>(a, tc.d);
            *name = "eval_team_kernel";
            return cudaGetLastError();
        }
    }
    if (uses_pair(a.n)) {
        const PairChoice tc = pair_choice(a.n, nsp);
        if (tc.d.smem_bytes <= (size_t)smem_optin && tc.d.C >= nsp) {
            int per_sm = 1;
            cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tc.fn, tc.d.threads, tc.d.smem_bytes);
            if (e != cudaSuccess) return e;
            if (per_sm < 1) per_sm = 1;
            const long long teams = (a.batch * nsp + tc.d.C - 1) / tc.d.C;
            long long grid = (long long)num_sms * per_sm;
            if (grid > teams) grid = teams;
            tc.fn<<<(unsigned)grid, tc.d.threads, tc.d.smem_bytes, stream>>>(a, tc.d);
            *name = "eval_pair_kernel";
            return cudaGetLastError();
        }
    }
    if (a.fused) return cudaErrorInvalidValue;   // only the team and pair kernels assemble G on the fly
    if (uses_pair_global(a.n, nsp) && a.scratch != nullptr) {
        const PairChoice tc = pair_global_choice(a.n, nsp);
        if (tc.d.smem_bytes <= (size_t)smem_optin && (size_t)tc.d.rec_doubles <= a.scratch_stride) {
            int per_sm = 1;
            cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tc.fn, tc.d.threads, tc.d.smem_bytes);
            if (e != cudaSuccess) return e;
            if (per_sm < 1) per_sm = 1;
            long long grid = (long long)num_sms * per_sm;
            const long long cap = eval_max_ctas(a.n, a.batch, num_sms, smem_optin);
            if (grid > cap) grid = cap;
            if (grid > a.batch) grid = a.batch;            // one configuration (C / nsp) per team
            tc.fn<<<(unsigned)grid, tc.d.threads, tc.d.smem_bytes, stream>>>(a, tc.d);
            *name = "eval_pair_kernel(global)";
            return cudaGetLastError();
        }
    }
    if (uses_big(a.n)) {
        const TiledDims d = big_dims(a.n, nsp);
        const size_t smem = (size_t)d.tab_bytes;
        int per_sm = 1;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, big_kernel(), kBigThreads, smem);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) per_sm = 1;
        long long grid = (long long)num_sms * per_sm;
        const long long cap = eval_max_ctas(a.n, a.batch, num_sms, smem_optin);
        if (grid > cap) grid = cap;
        big_kernel()<<<(unsigned)grid, kBigThreads, smem, stream>>>(a, d);
        *name = "eval_tiled_kernel(global)";
        return cudaGetLastError();
    }
    const int G = tiled_group(a.n, nsp, smem_optin);
    if (G > 0) {
        const TiledDims d = tiled_dims<kTiledB>(a.n, G, nsp);
        const size_t smem = tiled_smem_bytes<kTiledB>(a.n, G, nsp);
        int per_sm = 1;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tiled_kernel(), kTiledThreads, smem);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) per_sm = 1;
        const long long groups = (a.batch + G - 1) / G;
        long long grid = (long long)num_sms * per_sm;
        if (grid > groups) grid = groups;
        tiled_kernel()<<<(unsigned)grid, kTiledThreads, smem, stream>>>(a, d);
        *name = "eval_tiled_kernel";
        return cudaGetLastError();
    }
    const bool use_global = generic_needs_global(a.n, smem_optin);
    const size_t smem = use_global ? sizeof(double) * generic_small_doubles(a.n) : generic_smem_bytes(a.n, nsp);
    int per_sm = 1;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, eval_generic_kernel<kGenericThreads>,
                                                                  kGenericThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long grid = (long long)num_sms * per_sm;
    if (use_global) {
        const long long cap = eval_max_ctas(a.n, a.batch, num_sms, smem_optin);
        if (grid > cap) grid = cap;
    }
    if (grid > a.batch) grid = a.batch;
    eval_generic_kernel<kGenericThreads><<<(unsigned)grid, kGenericThreads, smem, stream>>>(a, nsp, use_global ? 1 : 0);
    *name = "eval_generic_kernel";
    return cudaGetLastError();
}

}  // namespace cosb
