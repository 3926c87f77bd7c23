// cos_dispatch.cuh -- picks the kernel variant for an evaluation launch and sizes its resources.
#pragma once
#include "cos_common.cuh"
#include "cos_kernels_generic.cuh"

namespace cosb {

constexpr int kGenericThreads = 256;

inline size_t generic_smem_bytes(int n, int nsp)
{
    return sizeof(double) * (generic_small_doubles(n) + ((size_t)nsp << n) + generic_frontier_doubles(n));
}

// True when the generic kernel must keep Z and the frontier in global scratch.
inline bool generic_needs_global(int n, int smem_optin)
{
    return generic_smem_bytes(n, 2) > (size_t)smem_optin;
}

// Doubles of global scratch per CTA (0: everything lives in shared memory).
inline size_t eval_scratch_doubles(int n, int smem_optin)
{
    if (!generic_needs_global(n, smem_optin)) return 0;
    return ((size_t)2 << n) + generic_frontier_doubles(n);
}

inline int eval_max_ctas(int n, long long batch, int num_sms, int smem_optin)
{
    (void)n; (void)smem_optin;
    const long long cap = (long long)num_sms * 2;
    return (int)(batch < cap ? batch : cap);
}

inline cudaError_t configure_kernels(int smem_optin)
{
    return cudaFuncSetAttribute(eval_generic_kernel<kGenericThreads>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
}

inline cudaError_t dispatch_eval(const EvalArgs& a, cudaStream_t stream, int num_sms, int smem_optin,
                                 int* launches, const char** name)
{
    const int nsp = (a.Gdn == a.Gup) ? 1 : 2;
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
    *launches = 1;
    *name = "eval_generic_kernel";
    return cudaGetLastError();
}

}  // namespace cosb
