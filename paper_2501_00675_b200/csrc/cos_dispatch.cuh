// cos_dispatch.cuh -- picks the kernel variant for an evaluation launch and sizes its resources.
//   n = 1..4                        eval_generic_kernel   (one thread per node, frontier in shared memory)
//   n = 5..10                       eval_team_kernel      (C instances per CTA, thread-bit register tiles)
//   n = 11..16                      eval_pair_kernel      (items split over lane pairs, records in per-CTA global
//                                   scratch, teams of 1..16 instances per CTA chosen by pair_plan)
// The FP32 entry points dispatch the same kernels from namespace f32 (float records).
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
    if (n == 9) return {f32::eval_team_kernel<8, 160, 4>, f32::team_dims<8>(n, nsp)};
    if (n == 8) return {f32::eval_team_kernel<16, 160, 4>, f32::team_dims<16>(n, nsp)};
    return {f32::eval_team_kernel<32, 192, 2>, f32::team_dims<32>(n, nsp)};
}

// ---- pair kernel (orders 11..16): the team mapping with every item split over a lane pair ----
// The records (Z, frontier, reduction arrays) live in a per-CTA block of global scratch served by L1/L2, so a CTA is
// not limited by the 227 KB of an SM and works on a TEAM of several instances: every level then exposes that many
// times more items per block barrier.  Measured (round 2, product build, kernel ms, column windows of 8 -- the
// windows of 6 adopted later take another 5-10 % off every figure; "shared" = the round-1 kernel with the records
// in shared memory, since removed):
//   one species  n=11: shared 0.221, C=8 0.226, C=16 0.216   n=12: shared 0.549, C=4 0.501, C=8 0.490, C=16 0.538
//                n=13: shared 0.388, C=1 0.42, C=2 0.361, C=4 0.333, C=8 0.355   n=14: C=1 0.864, C=2 0.846, C=4 0.855
//                n=15: C=1 1.214, C=2 1.107, C=4 1.126        n=16 (batch 256): C=1 1.740, C=2 1.577
//   two species  n=11: shared 0.376, C=8 0.348, C=16 0.327   n=12: shared 0.973, C=4 0.809, C=8 0.684
//                n=13: C=2 0.571, C=4 0.480, C=8 0.511        n=15: C=2 1.705, C=4 1.500    n=16: C=2 2.280, C=4 1.992
//   FP32         n=11: C=8 0.153, C=16 0.128   n=12: C=8 0.294, C=16 0.285   n=13: C=4 0.210, C=8 0.179   n=14: C=4 0.517
constexpr int kPairMinN = 11, kPairThreads = 512;
struct PairPlan {
    int C;           // instances per team
    bool red_smem;   // reduction arrays in shared memory instead of the scratch block
    bool small;      // two CTAs of 256 threads per SM instead of one of 512
};
// The plan of one launch: how many instances a CTA takes at a time.
inline PairPlan pair_plan(int n, int nsp, long long batch, int num_sms, bool f32)
{
    PairPlan p{2, false, false};
    if (!f32) {
        if (n == 11) p = (nsp == 1) ? PairPlan{8, false, true} : PairPlan{16, false, false};   // one species: two CTAs of 256
                                           // threads with teams of 8: 0.203 ms against 0.216 (one CTA of 512, teams of 16)
        else if (n == 12) p.C = 8;
        else if (n == 13) p.C = 4;
        else if (n == 14) p = (nsp == 1) ? PairPlan{1, true, false} : PairPlan{2, false, false};   // one instance: its reduction arrays
                                                                    // (128 KB) fit in shared memory: 0.813 against 0.844 ms
        else p.C = (nsp == 1) ? 2 : 4;
    } else {                           // float records: half the L1/L2 traffic, larger teams pay off
        p.C = n <= 12 ? 16 : (n == 13 ? 8 : 4);
    }
    // shrink the team only when more than half of the SMs would get no team at all
    // (n = 16, batch 256: 128 teams of 2 on 148 SMs measured 1.58 ms against 1.74 ms for 256 teams of 1)
    while (p.C > nsp && (batch * nsp + p.C - 1) / p.C < num_sms / 2) { p.C /= 2; p.red_smem = false; p.small = false; }
    return p;
}

// Precision traits: the same launch table serves cosb::f64 and cosb::f32.
struct Prec64 {
    static constexpr bool kF32 = false;
    using Dims = f64::PairDims;
    template <int C> static auto kernel() { return f64::eval_pair_kernel<C, kPairThreads, 1, 6>; }
    template <int C> static auto kernel_small() { return f64::eval_pair_kernel<C, kPairThreads / 2, 2, 6>; }
    template <int C> static Dims dims(int n, int nsp, bool rs, int threads = kPairThreads) { return f64::pair_dims<C>(n, threads, nsp, rs); }
};
struct Prec32 {
    static constexpr bool kF32 = true;
    using Dims = f32::PairDims;
    template <int C> static auto kernel() { return f32::eval_pair_kernel<C, kPairThreads, 1, 6>; }
    template <int C> static auto kernel_small() { return f32::eval_pair_kernel<C, kPairThreads / 2, 2, 6>; }
    template <int C> static Dims dims(int n, int nsp, bool rs, int threads = kPairThreads) { return f32::pair_dims<C>(n, threads, nsp, rs); }
};

// Calls f(kernel, dims) for the kernel instance of plan p at order n (false: no such instance).
template <class P, class F>
inline bool with_pair_instance(const PairPlan& p, int n, int nsp, F&& f)
{
    if (p.small) {
        if (p.C != 8) return false;
        f(P::template kernel_small<8>(), P::template dims<8>(n, nsp, p.red_smem, kPairThreads / 2));
        return true;
    }
    switch (p.C) {
        case 1: f(P::template kernel<1>(), P::template dims<1>(n, nsp, p.red_smem)); return true;
        case 2: f(P::template kernel<2>(), P::template dims<2>(n, nsp, p.red_smem)); return true;
        case 4: f(P::template kernel<4>(), P::template dims<4>(n, nsp, p.red_smem)); return true;
        case 8: f(P::template kernel<8>(), P::template dims<8>(n, nsp, p.red_smem)); return true;
        case 16: f(P::template kernel<16>(), P::template dims<16>(n, nsp, p.red_smem)); return true;
        default: return false;
    }
}

// Elements of global scratch per CTA for plan p.
template <class P>
inline size_t pair_plan_scratch(const PairPlan& p, int n, int nsp)
{
    size_t v = 0;
    with_pair_instance<P>(p, n, nsp, [&](auto, const typename P::Dims& d) { v = (size_t)d.rec_doubles; });
    return v;
}

// Elements of global scratch per CTA (0: everything lives in shared memory).
inline size_t eval_scratch_doubles(int n, int nsp, long long batch, int num_sms, int smem_optin, bool force_generic, bool f32)
{
    if (force_generic) return generic_scratch_doubles(n, smem_optin);
    if (n < kPairMinN) return 0;
    const PairPlan p = pair_plan(n, nsp, batch, num_sms, f32);
    return f32 ? pair_plan_scratch<Prec32>(p, n, nsp) : pair_plan_scratch<Prec64>(p, n, nsp);
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
    // every pair-kernel instance the plans can name: the attribute is set on first use (launch_pair), see below
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

// Launches the pair-kernel instance plan p names, on the configurations [0, a.batch) of `a`.  The opt-in shared-memory
// attribute of an instance is set when it is used (a handful of instances per precision; setting it again is harmless).
template <class P>
inline cudaError_t launch_pair_plan(const EvalArgs& a, const PairPlan& p, int nsp, int num_sms, int smem_optin,
                                    cudaStream_t stream)
{
    cudaError_t err = cudaErrorInvalidValue;
    const bool found = with_pair_instance<P>(p, a.n, nsp, [&](auto fn, const typename P::Dims& d) {
        if (a.scratch == nullptr || (size_t)d.rec_doubles > a.scratch_stride) return;
        if (d.smem_bytes > (size_t)smem_optin) return;
        err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (err != cudaSuccess) return;
        const long long teams = (a.batch * nsp + d.C - 1) / d.C;
        err = launch_persistent(fn, d, a, teams, eval_max_ctas(a.batch, num_sms), num_sms, stream);
    });
    return found ? err : cudaErrorInvalidValue;
}

// The tail of a batch.  A persistent grid works in rounds of one team per CTA; when the last round would occupy at most
// half of the CTAs, its configurations are launched separately with the smallest team that still takes one round: a
// round lasts about as long as its team is large (n = 12, batch 4096, teams of 8 on 148 CTAs: 3.46 rounds cost 4;
// 3 rounds of 8 + 1 round of 4 cost 3.6).  Returns the number of configurations to run with plan p; *tail gets the
// plan of the rest (tail->C == 0: no split).
inline long long pair_tail_split(const PairPlan& p, int nsp, long long batch, int num_sms, PairPlan* tail)
{
    tail->C = 0; tail->red_smem = false; tail->small = false;
    if (p.small || p.C / 2 < nsp) return batch;
    const long long grid = num_sms;                                  // one CTA of 512 threads per SM
    const long long teams = (batch * nsp + p.C - 1) / p.C;
    const long long full = teams / grid, rem = teams - full * grid;
    if (full < 1 || rem == 0 || rem > grid / 2) return batch;
    const long long head = full * grid * p.C / nsp;                  // configurations of the full rounds
    int c = p.C / 2;
    while (c / 2 >= nsp && ((batch - head) * nsp + c / 2 - 1) / (c / 2) <= grid) c /= 2;
    tail->C = c;
    return head;
}

template <class P>
inline cudaError_t launch_pair(const EvalArgs& a, int nsp, int num_sms, int smem_optin, cudaStream_t stream,
                               const char** name, const char* kernel_name, int* launches)
{
    *name = kernel_name;
    const PairPlan plan = pair_plan(a.n, nsp, a.batch, num_sms, P::kF32);
    PairPlan tail;
    const long long head = pair_tail_split(plan, nsp, a.batch, num_sms, &tail);
    if (tail.C == 0) return launch_pair_plan<P>(a, plan, nsp, num_sms, smem_optin, stream);
    EvalArgs h = a, t = a;
    h.batch = head;
    t.batch = a.batch - head;
    const size_t es = P::kF32 ? sizeof(float) : sizeof(double);     // element size behind the input pointers
    const size_t go = (size_t)head * a.n * a.n * es, uo = (size_t)head * a.n * es;
    t.Gup = reinterpret_cast<const double*>(reinterpret_cast<const char*>(a.Gup) + go);
    t.Gdn = reinterpret_cast<const double*>(reinterpret_cast<const char*>(a.Gdn) + go);
    if (a.u) t.u = reinterpret_cast<const double*>(reinterpret_cast<const char*>(a.u) + uo);
    t.out = a.out + head;
    cudaError_t e = launch_pair_plan<P>(h, plan, nsp, num_sms, smem_optin, stream);
    if (e != cudaSuccess) return e;
    *launches = 2;
    return launch_pair_plan<P>(t, tail, nsp, num_sms, smem_optin, stream);
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
    if (!force_generic && a.n >= kPairMinN) {
        return launch_pair<Prec64>(a, nsp, num_sms, smem_optin, stream, name, "eval_pair_kernel", launches);
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
inline cudaError_t dispatch_eval_f32(const EvalArgs& a, cudaStream_t stream, int num_sms, int smem_optin, int* launches,
                                     const char** name)
{
    const int nsp = (a.Gdn == a.Gup) ? 1 : 2;
    *launches = 1;
    if (uses_team(a.n)) {
        const TeamChoice32 tc = team_choice_f32(a.n, nsp);
        *name = "eval_team_kernel<float>";
        return launch_persistent(tc.fn, tc.d, a, (a.batch * nsp + tc.d.C - 1) / tc.d.C, 0, num_sms, stream);
    }
    if (a.n >= kPairMinN)
        return launch_pair<Prec32>(a, nsp, num_sms, smem_optin, stream, name, "eval_pair_kernel<float>", launches);
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
