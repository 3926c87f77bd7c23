// cos_dispatch.cuh -- picks the kernel variant for an evaluation launch and sizes its resources.
//   n = 1..4                        eval_generic_kernel   (one thread per node, frontier in shared memory)
//   n = 5..10                       eval_team_kernel      (C instances per CTA, thread-bit register tiles)
//   n = 11..13 (one species <= 13,
//               two species <= 12)  eval_pair_kernel      (items split over lane pairs, shared memory)
//   n = 14..16, two species n = 13  eval_pair_kernel<..., GLOBAL = true>  (records in per-CTA global scratch)
// The FP32 entry points dispatch the same shapes from namespace f32 (float records).
// The generic kernel also runs any order when the context is told to (cos_debug_force_generic): it is the
// in-library cross-check of the tuned kernels, not a fallback for another device.
#pragma once
#include "cos_common.cuh"
#include "cos_kernels_generic.cuh"
#include "cos_kernels_typed.cuh"

namespace cosb {

constexpr int kGenericThreads = 256;

inline size_t generic_smem_bytes(int n, int nsp, size_t elem = sizeof(double))
{
    return elem * (generic_small_doubles(n) + ((size_t)nsp << n) + generic_frontier_doubles(n));
}

// True when the generic kernel must keep Z and the frontier in global scratch.
inline bool generic_needs_global(int n, int smem_optin)
{
    return generic_smem_bytes(n, 2) > (size_t)smem_optin;
}

inline size_t generic_scratch_doubles(int n, int smem_optin)
{
    return generic_needs_global(n, smem_optin) ? ((size_t)2 << n) + generic_frontier_doubles(n) : 0;
}

// ---- team kernel (orders 5..10): instances per team and launch shape per order ----
constexpr int kTeamMinN = 5, kTeamMaxN = 10;
using TeamKernel = void (*)(EvalArgs, f64::TeamDims);
struct TeamChoice { TeamKernel fn; f64::TeamDims d; };
inline bool uses_team(int n) { return n >= kTeamMinN && n <= kTeamMaxN; }
inline TeamChoice team_choice(int n, int nsp)
{
    if (n == 10) return {f64::eval_team_kernel<4, 160, 2>, f64::team_dims<4>(n, nsp)};
    if (n == 9) return {f64::eval_team_kernel<8, 160, 2>, f64::team_dims<8>(n, nsp)};
    if (n == 8) return {f64::eval_team_kernel<16, 160, 2>, f64::team_dims<16>(n, nsp)};
    return {f64::eval_team_kernel<32, 192, 2>, f64::team_dims<32>(n, nsp)};
}
// FP32 variant: the same kernels instantiated for float; half the shared memory per instance, so
// more teams are resident per SM (the launch bounds only cap the registers)
using TeamKernel32 = void (*)(EvalArgs, f32::TeamDims);
struct TeamChoice32 { TeamKernel32 fn; f32::TeamDims d; };
inline TeamChoice32 team_choice_f32(int n, int nsp)
{
    if (n == 10) return {f32::eval_team_kernel<4, 160, 3>, f32::team_dims<4>(n, nsp)};
    if (n == 9) return {f32::eval_team_kernel<8, 160, 3>, f32::team_dims<8>(n, nsp)};
    if (n == 8) return {f32::eval_team_kernel<16, 160, 3>, f32::team_dims<16>(n, nsp)};
    return {f32::eval_team_kernel<32, 192, 2>, f32::team_dims<32>(n, nsp)};
}

// ---- pair kernel (orders 11..13): the team mapping with every item split over a lane pair ----
constexpr int kPairMinN = 11, kPairMaxN = 13;
using PairKernel = void (*)(EvalArgs, f64::PairDims);
struct PairChoice { PairKernel fn; f64::PairDims d; };
using PairKernel32 = void (*)(EvalArgs, f32::PairDims);
struct PairChoice32 { PairKernel32 fn; f32::PairDims d; };
inline bool uses_pair(int n, int nsp) { return n >= kPairMinN && n <= (nsp == 1 ? kPairMaxN : kPairMaxN - 1); }
inline PairChoice pair_choice(int n, int nsp)
{
    if (n == 13) return {f64::eval_pair_kernel<1, 512, 1, 10>, f64::pair_dims<1>(n, 1)};   // one species only
    if (n == 12) return {f64::eval_pair_kernel<2, 512, 1, 9>, f64::pair_dims<2>(n, nsp)};
    return {f64::eval_pair_kernel<4, 512, 1, 8>, f64::pair_dims<4>(n, nsp, 512)};
}
inline PairChoice32 pair_choice_f32(int n, int nsp)       // float records: twice the instances fit
{
    if (n == 13) return {f32::eval_pair_kernel<2, 512, 1, 10>, f32::pair_dims<2>(n, nsp, 512)};
    if (n == 12) return {f32::eval_pair_kernel<4, 512, 1, 9>, f32::pair_dims<4>(n, nsp, 512)};
    return {f32::eval_pair_kernel<4, 512, 1, 8>, f32::pair_dims<4>(n, nsp, 512)};
}

// ---- pair kernel on global records (orders 14..16; two species from 13): Z / frontier / reduction arrays in L2 scratch ----
constexpr int kPairGlobalMinN = 14, kPairGlobalThreads = 512;
inline bool uses_pair_global(int n, int nsp)
{
    return n <= kMaxN && (nsp == 1 ? n >= kPairGlobalMinN : n >= kPairGlobalMinN - 1);
}
inline PairChoice pair_global_choice(int n, int nsp = 1)
{
    if (nsp == 2) return {f64::eval_pair_kernel<2, kPairGlobalThreads, 1, 8, true>, f64::pair_dims_global<2>(n, kPairGlobalThreads, 2)};
    return {f64::eval_pair_kernel<1, kPairGlobalThreads, 1, 8, true>, f64::pair_dims_global<1>(n, kPairGlobalThreads)};
}
inline PairChoice32 pair_global_choice_f32(int n, int nsp = 1)
{
    if (nsp == 2) return {f32::eval_pair_kernel<2, kPairGlobalThreads, 1, 8, true>, f32::pair_dims_global<2>(n, kPairGlobalThreads, 2)};
    return {f32::eval_pair_kernel<1, kPairGlobalThreads, 1, 8, true>, f32::pair_dims_global<1>(n, kPairGlobalThreads)};
}
inline size_t pair_global_rec_doubles(int n)
{
    if (n < kPairGlobalMinN - 1 || n > kMaxN) return 0;
    const size_t a = (size_t)pair_global_choice(n, 1).d.rec_doubles, b = (size_t)pair_global_choice(n, 2).d.rec_doubles;
    return a > b ? a : b;
}

// Doubles of global scratch per CTA (0: everything lives in shared memory).
inline size_t eval_scratch_doubles(int n, int smem_optin, bool force_generic)
{
    if (force_generic) return generic_scratch_doubles(n, smem_optin);
    return pair_global_rec_doubles(n);
}

inline int eval_max_ctas(long long batch, int num_sms)
{
    const long long cap = (long long)num_sms * 2;
    return (int)(batch < cap ? batch : cap);
}

inline cudaError_t configure_kernels(int smem_optin)
{
    cudaError_t e = cudaFuncSetAttribute(f64::eval_generic_kernel<kGenericThreads>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(f32::eval_generic_kernel<kGenericThreads>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
    for (int n = kTeamMinN; n <= kTeamMaxN; ++n) {
        e = cudaFuncSetAttribute(team_choice(n, 1).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(team_choice_f32(n, 1).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (e != cudaSuccess) return e;
    }
    for (int n = kPairMinN; n <= kPairMaxN; ++n) {
        e = cudaFuncSetAttribute(pair_choice(n, 1).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(pair_choice_f32(n, 1).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (e != cudaSuccess) return e;
    }
    for (int nsp = 1; nsp <= 2; ++nsp) {
        e = cudaFuncSetAttribute(pair_global_choice(kPairGlobalMinN, nsp).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(pair_global_choice_f32(kPairGlobalMinN, nsp).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

template <class Kernel, class Dims>
inline cudaError_t launch_persistent(Kernel fn, const Dims& d, const EvalArgs& a, long long teams, long long cap,
                                     int num_sms, cudaStream_t stream)
{
    int per_sm = 1;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, d.threads, d.smem_bytes);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long grid = (long long)num_sms * per_sm;
    if (grid > teams) grid = teams;
    if (cap > 0 && grid > cap) grid = cap;
    fn<<<(unsigned)grid, d.threads, d.smem_bytes, stream>>>(a, d);
    return cudaGetLastError();
}

inline cudaError_t dispatch_eval(const EvalArgs& a, cudaStream_t stream, int num_sms, int smem_optin,
                                 bool force_generic, int* launches, const char** name)
{
    const int nsp = (a.Gdn == a.Gup) ? 1 : 2;
    *launches = 1;
    if (!force_generic && uses_team(a.n)) {
        const TeamChoice tc = team_choice(a.n, nsp);
        *name = "eval_team_kernel";
        return launch_persistent(tc.fn, tc.d, a, (a.batch * nsp + tc.d.C - 1) / tc.d.C, 0, num_sms, stream);
    }
    if (!force_generic && uses_pair(a.n, nsp)) {
        const PairChoice tc = pair_choice(a.n, nsp);
        *name = "eval_pair_kernel";
        return launch_persistent(tc.fn, tc.d, a, (a.batch * nsp + tc.d.C - 1) / tc.d.C, 0, num_sms, stream);
    }
    if (!force_generic && uses_pair_global(a.n, nsp)) {
        const PairChoice tc = pair_global_choice(a.n, nsp);
        if (a.scratch == nullptr || (size_t)tc.d.rec_doubles > a.scratch_stride) return cudaErrorInvalidValue;
        *name = "eval_pair_kernel(global)";
        return launch_persistent(tc.fn, tc.d, a, a.batch, eval_max_ctas(a.batch, num_sms), num_sms, stream);
    }
    const bool use_global = generic_needs_global(a.n, smem_optin);
    if (use_global && a.scratch == nullptr) return cudaErrorInvalidValue;
    const size_t smem = use_global ? sizeof(double) * generic_small_doubles(a.n) : generic_smem_bytes(a.n, nsp);
    int per_sm = 1;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, f64::eval_generic_kernel<kGenericThreads>,
                                                                  kGenericThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long grid = (long long)num_sms * per_sm;
    if (use_global) {
        const long long cap = eval_max_ctas(a.batch, num_sms);
        if (grid > cap) grid = cap;
    }
    if (grid > a.batch) grid = a.batch;
    f64::eval_generic_kernel<kGenericThreads><<<(unsigned)grid, kGenericThreads, smem, stream>>>(a, nsp, use_global ? 1 : 0);
    *name = "eval_generic_kernel";
    return cudaGetLastError();
}

// FP32 variant: orders 1..4 on the plain kernel, 5..10 on the team kernel, both instantiated for float.  The input
// pointers of `a` address FP32 copies of G and u (made by the entry point).
inline cudaError_t dispatch_eval_f32(const EvalArgs& a, cudaStream_t stream, int num_sms, int* launches, const char** name)
{
    const int nsp = (a.Gdn == a.Gup) ? 1 : 2;
    *launches = 1;
    if (uses_team(a.n)) {
        const TeamChoice32 tc = team_choice_f32(a.n, nsp);
        *name = "eval_team_kernel<float>";
        return launch_persistent(tc.fn, tc.d, a, (a.batch * nsp + tc.d.C - 1) / tc.d.C, 0, num_sms, stream);
    }
    if (uses_pair(a.n, nsp)) {
        const PairChoice32 tc = pair_choice_f32(a.n, nsp);
        *name = "eval_pair_kernel<float>";
        return launch_persistent(tc.fn, tc.d, a, (a.batch * nsp + tc.d.C - 1) / tc.d.C, 0, num_sms, stream);
    }
    if (uses_pair_global(a.n, nsp)) {
        const PairChoice32 tc = pair_global_choice_f32(a.n, nsp);
        if (a.scratch == nullptr || (size_t)tc.d.rec_doubles > a.scratch_stride) return cudaErrorInvalidValue;
        *name = "eval_pair_kernel<float>(global)";
        return launch_persistent(tc.fn, tc.d, a, a.batch, eval_max_ctas(a.batch, num_sms), num_sms, stream);
    }
    const size_t smem = generic_smem_bytes(a.n, nsp, sizeof(float));
    int per_sm = 1;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, f32::eval_generic_kernel<kGenericThreads>,
                                                                  kGenericThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long grid = (long long)num_sms * per_sm;
    if (grid > a.batch) grid = a.batch;
    f32::eval_generic_kernel<kGenericThreads><<<(unsigned)grid, kGenericThreads, smem, stream>>>(a, nsp, 0);
    *name = "eval_generic_kernel<float>";
    return cudaGetLastError();
}

}  // namespace cosb
