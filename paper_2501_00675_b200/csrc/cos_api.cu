// cos_api.cu -- C-ABI entry points of libcos_b200.so (include/cos.h): context, argument validation,
// scratch management, kernel dispatch.  Host code only touches pointers and sizes; every step of the
// path (a1..a5) runs in the kernels.  There is no CPU fallback.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "cos_common.cuh"
#include "cos_internal.h"
#include "cos_dispatch.cuh"
#include "cos_mc.cuh"

using namespace cosb;

struct cos_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    int smem_optin = 0;
    // G0 tables (borrowed)
    const double* table[2] = {nullptr, nullptr};
    int Lx = 0, Ly = 0, ntau = 0;
    double beta = 0.0;
    // scratch (owned)
    uint32_t* off = nullptr;
    double* scratch = nullptr;      size_t scratch_bytes = 0;
    double* gscratch = nullptr;     size_t gscratch_bytes = 0;   // G matrices of cos_eval_connected_xt
    unsigned char* team_tabs[COS_MAX_ORDER + 1] = {};            // per order: table image of the team kernel / item
                                                                 // descriptors of the pair kernel
    void* stage = nullptr;          size_t stage_bytes = 0;      // device staging of the host path
    unsigned char* team_tabs32[COS_MAX_ORDER + 1] = {};          // FP32 variant: table images of the team kernel
    float* g32 = nullptr;           size_t g32_bytes = 0;        // FP32 variant: converted copies of G_up, G_down, u
    void* mc = nullptr;             size_t mc_bytes = 0;         // cos_mc_run: proposal coordinates and weights
    unsigned char* noalloc_scratch = nullptr;                    // device address of g_noalloc_scratch on this device
    cudaStream_t copy_stream = nullptr;                          // host path: H2D of chunk k+1 behind the kernels of chunk k
    cudaEvent_t copy_done[2] = {nullptr, nullptr};
    // bookkeeping
    double loop_weight = 1.0;       // N_f: every closed fermion loop contributes -N_f (cos_set_loop_weight)
    bool force_generic = false;     // cos_debug_force_generic: every order through eval_generic_kernel
    int last_launches = 0;
    const char* last_kernel = "none";
    cudaError_t last_err = cudaSuccess;
    // optional timing of the evaluation kernel
    bool timing = false;
    std::vector<cudaEvent_t> ev;    // pairs (start, stop)
    size_t ev_used = 0;
};

// Scratch of cos_eval_connected_noalloc (include/cos.h): item descriptors of the order, then the record blocks of the
// thread blocks.  One copy per GPU that loads the library, held until the process exits, shared by every call.  In host
// code this name is a host-side stand-in, never a device address: cos_create asks the runtime for the address on its
// device (cudaGetSymbolAddress) and the entry point passes that pointer to the kernels.
static __device__ __align__(256) unsigned char g_noalloc_scratch[COS_NOALLOC_SCRATCH_BYTES];

namespace {

int fail_cuda(cos_ctx* c, cudaError_t e)
{
    if (c) c->last_err = e;
    return COS_ECUDA;
}

#define COS_CUDA(c, expr)                                   \
    do {                                                    \
        cudaError_t e__ = (expr);                           \
        if (e__ != cudaSuccess) return fail_cuda((c), e__); \
    } while (0)

int grow(cos_ctx* c, void** p, size_t* have, size_t need)
{
    if (need <= *have) return COS_OK;
    if (*p) {
        COS_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(*p);
        *p = nullptr;
        *have = 0;
    }
    cudaError_t e = cudaMalloc(p, need);
    if (e != cudaSuccess) { c->last_err = e; (void)cudaGetLastError(); return COS_ENOMEM; }
    *have = need;
    return COS_OK;
}

int alloc_dev(cos_ctx* c, void** p, size_t bytes)
{
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) { c->last_err = e; (void)cudaGetLastError(); *p = nullptr; return COS_ENOMEM; }
    return COS_OK;
}

bool timer_begin(cos_ctx* c)
{
    if (!c->timing) return false;
    if (c->ev_used + 2 > c->ev.size()) {
        for (int k = 0; k < 2; ++k) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return false;
            c->ev.push_back(e);
        }
    }
    cudaEventRecord(c->ev[c->ev_used], c->stream);
    return true;
}
void timer_end(cos_ctx* c)
{
    cudaEventRecord(c->ev[c->ev_used + 1], c->stream);
    c->ev_used += 2;
}

int check_eval_args(cos_ctx* c, int n, long long batch, const void* gup, const void* gdn, const void* out)
{
    if (!c) return COS_EINVAL;
    if (n < 1 || n > COS_MAX_ORDER || batch < 0) return COS_EINVAL;
    if (batch > 0 && (!gup || !gdn || !out)) return COS_EINVAL;
    return COS_OK;
}

int launch_eval(cos_ctx* c, const EvalArgs& args)
{
    const bool t = timer_begin(c);
    int launches = 0;
    const char* name = nullptr;
    cudaError_t e = dispatch_eval(args, c->stream, c->num_sms, c->smem_optin, c->force_generic, &launches, &name);
    if (t) timer_end(c);
    if (e != cudaSuccess) return fail_cuda(c, e);
    c->last_launches += launches;
    c->last_kernel = name;
    return COS_OK;
}

int do_eval(cos_ctx* c, int n, long long batch, const double* gup, const double* gdn, const double* u,
            double U, double* out, int connected)
{
    if (batch == 0) return COS_OK;
    EvalArgs a{};
    a.n = n; a.batch = batch; a.Gup = gup; a.Gdn = gdn; a.u = u; a.U = U; a.out = out;
    a.connected = connected; a.off = c->off; a.loopf = -c->loop_weight;
    if (c->force_generic) {
        // no tables: the generic kernel computes its indices on the fly
    } else if (uses_team(n)) {   // table image of this order, built on first use
        if (!c->team_tabs[n]) {
            const f64::TeamDims td = team_choice(n, 1).d;
            unsigned char* buf = nullptr;
            if (alloc_dev(c, (void**)&buf, (size_t)td.tab_bytes) != COS_OK) return COS_ENOMEM;
            f64::team_tables_kernel<<<1, 256, (size_t)td.tab_bytes, c->stream>>>(td, buf);
            COS_CUDA(c, cudaGetLastError());
            c->team_tabs[n] = buf;
        }
        a.tabs = c->team_tabs[n];
    } else if (n >= kPairMinN) {   // item descriptors of the global-record pair kernel, built on first use
        if (!c->team_tabs[n]) {
            const size_t bytes = ((size_t)1 << (n - f64::kPairB)) * f64::kPairDscWords * sizeof(uint32_t);
            unsigned char* buf = nullptr;
            if (alloc_dev(c, (void**)&buf, bytes) != COS_OK) return COS_ENOMEM;
            f64::pair_tables_kernel<<<32, 256, 0, c->stream>>>(n, reinterpret_cast<uint32_t*>(buf));
            COS_CUDA(c, cudaGetLastError());
            c->team_tabs[n] = buf;
        }
        a.tabs = c->team_tabs[n];
    }
    // global scratch for the orders whose frontier does not fit in shared memory
    const size_t per_cta = eval_scratch_doubles(n, gdn == gup ? 1 : 2, batch, c->num_sms, c->smem_optin, c->force_generic, false);
    if (per_cta) {
        const int ctas = eval_max_ctas(batch, c->num_sms);
        int rc = grow(c, (void**)&c->scratch, &c->scratch_bytes, per_cta * sizeof(double) * (size_t)ctas);
        if (rc != COS_OK) return rc;
        a.scratch = c->scratch;
        a.scratch_stride = per_cta;
    }
    return launch_eval(c, a);
}

// FP32 variant, input side: one warp per configuration.  Every term of the result is homogeneous of degree 2n in
// the entries of G (n factors per species), so G is first scaled by a power of two s = 2^k (exact) that brings
// its root-mean-square entry to [1, 2): products of ten small Green's functions would otherwise leave the FP32
// range (cfg3: Z ~ 1e-20, D ~ Z^2 underflows).  The output kernel multiplies the result by 2^(-2nk).
__global__ void __launch_bounds__(256) convert_scale_f32_kernel(int n, long long batch, const double* __restrict__ gup,
                                                                const double* __restrict__ gdn, float* __restrict__ gu32,
                                                                float* __restrict__ gd32, int* __restrict__ kexp)
{
    const int lane = threadIdx.x & 31, nn = n * n;
    for (long long b = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5; b < batch;
         b += ((long long)gridDim.x * blockDim.x) >> 5) {
        const double* pu = gup + b * nn;
        const double* pd = gdn + b * nn;
        double ss = 0.0;
        for (int e = lane; e < nn; e += 32) { const double x = pu[e], y = pd[e]; ss += x * x + y * y; }
        for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
        int k = 0;
        if (ss > 0.0 && ss - ss == 0.0) k = -ilogb(sqrt(ss / (2.0 * nn)));      // rms * 2^k in [1, 2)
        const double sc = ldexp(1.0, k);
        for (int e = lane; e < nn; e += 32) {
            gu32[b * nn + e] = (float)(pu[e] * sc);                              // one rounding, to nearest even
            if (gd32 != gu32) gd32[b * nn + e] = (float)(pd[e] * sc);
        }
        if (lane == 0) kexp[b] = k;
    }
}

__global__ void __launch_bounds__(256) convert_f64_f32_kernel(const double* __restrict__ src, float* __restrict__ dst, size_t count)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < count; i += (size_t)gridDim.x * blockDim.x)
        dst[i] = (float)src[i];                       // round to nearest even
}

__global__ void __launch_bounds__(256) unscale_f32_kernel(int n, long long batch, const int* __restrict__ kexp, double* out)
{
    for (long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x; b < batch; b += (long long)gridDim.x * blockDim.x)
        out[b] = ldexp(out[b], -2 * n * kexp[b]);
}

// FP32 variant: G and u are rounded once to FP32, every later operation is FP32.
int do_eval_f32(cos_ctx* c, int n, long long batch, const double* gup, const double* gdn, const double* u, double U,
                double* out, int connected)
{
    if (batch == 0) return COS_OK;
    const bool two = gdn != gup;
    const size_t nn = (size_t)batch * n * n, nu = u ? (size_t)batch * n : 0;
    int rc = grow(c, (void**)&c->g32, &c->g32_bytes, sizeof(float) * ((two ? 2 : 1) * nn + nu) + sizeof(int) * (size_t)batch);
    if (rc != COS_OK) return rc;
    float* gu32 = c->g32;
    float* gd32 = two ? gu32 + nn : gu32;
    float* u32 = u ? gu32 + (two ? 2 : 1) * nn : nullptr;
    int* kexp = reinterpret_cast<int*>(gu32 + (two ? 2 : 1) * nn + nu);
    const unsigned blocks = (unsigned)c->num_sms * 8;
    convert_scale_f32_kernel<<<blocks, 256, 0, c->stream>>>(n, batch, gup, gdn, gu32, gd32, kexp);
    if (u) convert_f64_f32_kernel<<<blocks, 256, 0, c->stream>>>(u, u32, nu);
    COS_CUDA(c, cudaGetLastError());
    c->last_launches += 2 + (u ? 1 : 0);
    EvalArgs a{};
    a.n = n; a.batch = batch; a.U = U; a.out = out; a.connected = connected; a.off = c->off; a.loopf = -c->loop_weight;
    a.Gup = reinterpret_cast<const double*>(gu32);      // FP32 data behind the FP64-typed fields (read through in_real)
    a.Gdn = reinterpret_cast<const double*>(gd32);
    a.u = reinterpret_cast<const double*>(u32);
    if (uses_team(n)) {
        if (!c->team_tabs32[n]) {
            const f32::TeamDims td = team_choice_f32(n, 1).d;
            unsigned char* buf = nullptr;
            if (alloc_dev(c, (void**)&buf, (size_t)td.tab_bytes) != COS_OK) return COS_ENOMEM;
            f32::team_tables_kernel<<<1, 256, (size_t)td.tab_bytes, c->stream>>>(td, buf);
            COS_CUDA(c, cudaGetLastError());
            c->team_tabs32[n] = buf;
        }
        a.tabs = c->team_tabs32[n];
    } else if (n >= kPairMinN) {   // item descriptors of the global-record pair kernel (integers: shared with FP64)
        if (!c->team_tabs[n]) {
            const size_t bytes = ((size_t)1 << (n - f64::kPairB)) * f64::kPairDscWords * sizeof(uint32_t);
            unsigned char* buf = nullptr;
            if (alloc_dev(c, (void**)&buf, bytes) != COS_OK) return COS_ENOMEM;
            f64::pair_tables_kernel<<<32, 256, 0, c->stream>>>(n, reinterpret_cast<uint32_t*>(buf));
            COS_CUDA(c, cudaGetLastError());
            c->team_tabs[n] = buf;
        }
        a.tabs = c->team_tabs[n];
    }
    const size_t per_cta = eval_scratch_doubles(n, two ? 2 : 1, batch, c->num_sms, c->smem_optin, false, true);   // elements
    if (per_cta) {
        const int ctas = eval_max_ctas(batch, c->num_sms);
        rc = grow(c, (void**)&c->scratch, &c->scratch_bytes, per_cta * sizeof(double) * (size_t)ctas);
        if (rc != COS_OK) return rc;
        a.scratch = c->scratch;
        a.scratch_stride = per_cta;
    }
    const bool t = timer_begin(c);
    int launches = 0;
    const char* name = nullptr;
    cudaError_t e = dispatch_eval_f32(a, c->stream, c->num_sms, c->smem_optin, &launches, &name);
    if (t) timer_end(c);
    if (e != cudaSuccess) return fail_cuda(c, e);
    unscale_f32_kernel<<<blocks, 256, 0, c->stream>>>(n, batch, kexp, out);
    COS_CUDA(c, cudaGetLastError());
    c->last_launches += launches;
    c->last_kernel = name;
    return COS_OK;
}

int do_build_G(cos_ctx* c, int n, long long batch, const int* xy, const double* tau, double g_diag,
               double* gup, double* gdn)
{
    if (batch == 0) return COS_OK;
    BuildGArgs a{};
    a.n = n; a.batch = batch; a.xy = xy; a.tau = tau;
    a.Tup = c->table[0]; a.Tdn = c->table[1];
    a.Lx = c->Lx; a.Ly = c->Ly; a.ntau = c->ntau; a.beta = c->beta; a.g_diag = g_diag;
    a.Gup = gup; a.Gdn = (gdn == gup) ? nullptr : gdn;
    a.rbeta = 1.0 / c->beta;                                        // IEEE division: the correctly rounded reciprocal
    {
        unsigned long long bits;
        memcpy(&bits, &c->beta, sizeof bits);
        a.fast_div = (bits & 0xFFFFFFFFFFFFFull) != 0xFFFFFFFFFFFFFull;
    }
    long long blocks = (batch + kBuildGCfgs - 1) / kBuildGCfgs;     // configurations per CTA pass (see the kernel)
    const long long cap = (long long)c->num_sms * 8;
    if (blocks > cap) blocks = cap;
    build_G_kernel<<<(unsigned)blocks, build_G_threads(n), 0, c->stream>>>(a);
    COS_CUDA(c, cudaGetLastError());
    c->last_launches += 1;
    return COS_OK;
}

}  // namespace

extern "C" {

int cos_abi_version(void) { return COS_ABI_VERSION; }

const char* cos_strerror(int code)
{
    switch (code) {
        case COS_OK: return "success";
        case COS_EINVAL: return "invalid argument";
        case COS_ECUDA: return "CUDA error (see cos_last_cuda_error)";
        case COS_ENOMEM: return "device scratch allocation failed";
        case COS_ENOTABLE: return "G0 table not set (call cos_set_g0_table first)";
        case COS_ETOOBIG: return "order or batch beyond the fixed capacity of cos_eval_connected_noalloc (COS_NOALLOC_MAX_ORDER, COS_NOALLOC_MAX_BATCH)";
        default: return "unknown status";
    }
}

const char* cos_last_cuda_error(const cos_ctx* ctx)
{
    return ctx ? cudaGetErrorString(ctx->last_err) : "no context";
}

int cos_create(cos_ctx** out, int device, void* cuda_stream)
{
    if (!out) return COS_EINVAL;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
        (void)cudaGetLastError();
        return COS_ECUDA;
    }
    cos_ctx* c = new (std::nothrow) cos_ctx();
    if (!c) return COS_ENOMEM;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    if (cudaSetDevice(device) != cudaSuccess || cudaGetDeviceProperties(&prop, device) != cudaSuccess) {
        delete c;
        return COS_ECUDA;
    }
    if (prop.major != 10) {   // sm_100a only: no multi-backend dispatch, no fallback
        delete c;
        return COS_ECUDA;
    }
    c->num_sms = prop.multiProcessorCount;
    c->smem_optin = (int)prop.sharedMemPerBlockOptin;
    const uint32_t count_off = 1u << (COS_MAX_ORDER - 1);
    if (cudaMalloc((void**)&c->off, sizeof(uint32_t) * (count_off + 1)) != cudaSuccess) {
        delete c;
        return COS_ENOMEM;
    }
    init_off_table_kernel<<<1, 1024, 0, c->stream>>>(c->off, count_off + 1);
    cudaError_t e = configure_kernels(c->smem_optin);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) {   // address of the static scratch on THIS device (the device set above is current)
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        c->noalloc_scratch = static_cast<unsigned char*>(p);
    }
    if (e != cudaSuccess) {
        cudaFree(c->off);
        delete c;
        return COS_ECUDA;
    }
    *out = c;
    return COS_OK;
}

int cos_destroy(cos_ctx* c)
{
    if (!c) return COS_EINVAL;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    cudaFree(c->off);
    cudaFree(c->scratch);
    cudaFree(c->gscratch);
    cudaFree(c->stage);
    cudaFree(c->mc);
    cudaFree(c->g32);
    for (int i = 0; i <= COS_MAX_ORDER; ++i) cudaFree(c->team_tabs32[i]);
    for (int i = 0; i <= COS_MAX_ORDER; ++i) cudaFree(c->team_tabs[i]);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    for (cudaEvent_t e : c->copy_done) if (e) cudaEventDestroy(e);
    delete c;
    return COS_OK;
}

int cos_set_g0_table(cos_ctx* c, int spin, const double* d_table, int Lx, int Ly, int ntau, double beta)
{
    if (!c || !d_table || spin < -1 || spin > 1 || Lx < 1 || Ly < 1 || ntau < 2 || !(beta > 0.0)) return COS_EINVAL;
    if ((long long)Lx * Ly * ntau >= (1LL << 31)) return COS_EINVAL;      // table entries are indexed with 32 bits
    const bool other_set = (spin >= 0) && c->table[1 - spin] != nullptr;
    if (other_set && (Lx != c->Lx || Ly != c->Ly || ntau != c->ntau || beta != c->beta)) return COS_EINVAL;
    if (spin == -1) c->table[0] = c->table[1] = d_table;
    else c->table[spin] = d_table;
    c->Lx = Lx; c->Ly = Ly; c->ntau = ntau; c->beta = beta;
    return COS_OK;
}

int cos_build_G(cos_ctx* c, int n, long long batch, const int* d_xy, const double* d_tau, double g_diag,
                double* d_Gup, double* d_Gdn)
{
    if (!c || n < 1 || n > COS_MAX_ORDER || batch < 0) return COS_EINVAL;
    if (batch > 0 && (!d_xy || !d_tau || !d_Gup)) return COS_EINVAL;
    if (!c->table[0]) return COS_ENOTABLE;
    const bool single = (d_Gdn == nullptr || d_Gdn == d_Gup);
    if (!single && !c->table[1]) return COS_ENOTABLE;
    if (single && c->table[1] && c->table[1] != c->table[0]) return COS_EINVAL;  // one output, two tables
    cudaSetDevice(c->device);
    c->last_launches = 0;
    return do_build_G(c, n, batch, d_xy, d_tau, g_diag, d_Gup, single ? d_Gup : d_Gdn);
}

int cos_eval_all(cos_ctx* c, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                 const double* d_u, double U, double* d_out)
{
    int rc = check_eval_args(c, n, batch, d_Gup, d_Gdn, d_out);
    if (rc != COS_OK) return rc;
    cudaSetDevice(c->device);
    c->last_launches = 0;
    return do_eval(c, n, batch, d_Gup, d_Gdn, d_u, U, d_out, 0);
}

int cos_eval_connected(cos_ctx* c, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                       const double* d_u, double U, double* d_out)
{
    int rc = check_eval_args(c, n, batch, d_Gup, d_Gdn, d_out);
    if (rc != COS_OK) return rc;
    cudaSetDevice(c->device);
    c->last_launches = 0;
    return do_eval(c, n, batch, d_Gup, d_Gdn, d_u, U, d_out, 1);
}

int cos_eval_connected_noalloc(cos_ctx* c, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                               const double* d_u, double U, double* d_out)
{
    int rc = check_eval_args(c, n, batch, d_Gup, d_Gdn, d_out);
    if (rc != COS_OK) return rc;
    if (n > COS_NOALLOC_MAX_ORDER || batch > COS_NOALLOC_MAX_BATCH) return COS_ETOOBIG;
    if (n < COS_NOALLOC_MIN_ORDER) return COS_EINVAL;
    if (!c->noalloc_scratch) return COS_ECUDA;
    c->last_launches = 0;
    if (batch == 0) return COS_OK;
    COS_CUDA(c, cudaSetDevice(c->device));
    const int nsp = (d_Gdn == d_Gup) ? 1 : 2;
    // layout of the array: [item descriptors of order n, rounded up to 256 B][record blocks, one per thread block]
    const size_t dsc_bytes = (((size_t)1 << (n - f64::kPairB)) * f64::kPairDscWords * sizeof(uint32_t) + 255) & ~(size_t)255;
    const size_t cap_doubles = ((size_t)COS_NOALLOC_SCRATCH_BYTES - dsc_bytes) / sizeof(double);
    // the largest team, from the one cos_eval_connected would take downwards, whose records for a full grid fit
    PairPlan p = pair_plan(n, nsp, batch, c->num_sms, false);
    size_t per_cta = 0;
    long long grid_cap = 0;
    for (;;) {
        per_cta = pair_plan_scratch<Prec64>(p, n, nsp);
        if (per_cta == 0) return COS_EINVAL;
        const long long teams = (batch * nsp + p.C - 1) / p.C;
        long long grid = (long long)c->num_sms * (p.small ? 2 : 1);
        if (grid > teams) grid = teams;
        grid_cap = grid;
        if (per_cta * (size_t)grid <= cap_doubles) break;
        if (p.C / 2 >= nsp) { p = PairPlan{p.C / 2, false, false}; continue; }
        grid_cap = (long long)(cap_doubles / per_cta);      // smallest team: fewer thread blocks than SMs
        if (grid_cap < 1) return COS_ETOOBIG;
        break;
    }
    uint32_t* dsc = reinterpret_cast<uint32_t*>(c->noalloc_scratch);
    f64::pair_tables_kernel<<<32, 256, 0, c->stream>>>(n, dsc);
    COS_CUDA(c, cudaGetLastError());
    EvalArgs a{};
    a.n = n; a.batch = batch; a.Gup = d_Gup; a.Gdn = d_Gdn; a.u = d_u; a.U = U; a.out = d_out;
    a.connected = 1; a.off = c->off; a.loopf = -c->loop_weight;
    a.tabs = c->noalloc_scratch;
    a.scratch = reinterpret_cast<double*>(c->noalloc_scratch + dsc_bytes);
    a.scratch_stride = per_cta;
    cudaError_t err = cudaErrorInvalidValue;
    const int smem_optin = c->smem_optin, num_sms = c->num_sms;
    cudaStream_t stream = c->stream;
    // (not bracketed by the optional kernel timer: that would create events)
    const bool found = with_pair_instance<Prec64>(p, n, nsp, [&](auto fn, const Prec64::Dims& d) {
        if (d.smem_bytes > (size_t)smem_optin) return;
        err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
        if (err != cudaSuccess) return;
        err = launch_persistent(fn, d, a, (a.batch * nsp + d.C - 1) / d.C, grid_cap, num_sms, stream);
    });
    if (!found) return COS_EINVAL;
    if (err != cudaSuccess) return fail_cuda(c, err);
    c->last_launches = 2;
    c->last_kernel = "eval_pair_kernel (static scratch)";
    return COS_OK;
}

int cos_eval_all_f32(cos_ctx* c, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                     const double* d_u, double U, double* d_out)
{
    int rc = check_eval_args(c, n, batch, d_Gup, d_Gdn, d_out);
    if (rc != COS_OK) return rc;
    cudaSetDevice(c->device);
    c->last_launches = 0;
    return do_eval_f32(c, n, batch, d_Gup, d_Gdn, d_u, U, d_out, 0);
}

int cos_eval_connected_f32(cos_ctx* c, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                           const double* d_u, double U, double* d_out)
{
    int rc = check_eval_args(c, n, batch, d_Gup, d_Gdn, d_out);
    if (rc != COS_OK) return rc;
    cudaSetDevice(c->device);
    c->last_launches = 0;
    return do_eval_f32(c, n, batch, d_Gup, d_Gdn, d_u, U, d_out, 1);
}

int cos_eval_halfvertex(cos_ctx* c, int n_lines, long long batch, const double* d_W, const double* d_V, int connected,
                        double* d_out)
{
    if (!c || n_lines < 1 || 2 * n_lines > COS_MAX_ORDER || batch < 0) return COS_EINVAL;
    if (batch > 0 && (!d_W || !d_V || !d_out)) return COS_EINVAL;
    cudaSetDevice(c->device);
    c->last_launches = 0;
    if (batch == 0) return COS_OK;
    const int m = 2 * n_lines;
    EvalArgs a{};
    a.n = m; a.batch = batch; a.Gup = d_W; a.Gdn = d_W; a.u = d_V; a.U = 0.0; a.out = d_out;
    a.connected = connected != 0; a.off = c->off; a.loopf = -c->loop_weight; a.halfvertex = 1;
    const size_t per_cta = generic_scratch_doubles(m, c->smem_optin);
    if (per_cta) {
        const int ctas = eval_max_ctas(batch, c->num_sms);
        int rc = grow(c, (void**)&c->scratch, &c->scratch_bytes, per_cta * sizeof(double) * (size_t)ctas);
        if (rc != COS_OK) return rc;
        a.scratch = c->scratch;
        a.scratch_stride = per_cta;
    }
    const bool t = timer_begin(c);
    int launches = 0;
    const char* name = nullptr;
    cudaError_t e = dispatch_eval(a, c->stream, c->num_sms, c->smem_optin, /*force_generic=*/true, &launches, &name);
    if (t) timer_end(c);
    if (e != cudaSuccess) return fail_cuda(c, e);
    c->last_launches += launches;
    c->last_kernel = name;
    return COS_OK;
}

int cos_eval_connected_xt(cos_ctx* c, int n, long long batch, const int* d_xy, const double* d_tau,
                          double g_diag, const double* d_u, double U, double* d_out)
{
    if (!c || n < 1 || n > COS_MAX_ORDER || batch < 0) return COS_EINVAL;
    if (batch > 0 && (!d_xy || !d_tau || !d_out)) return COS_EINVAL;
    if (!c->table[0]) return COS_ENOTABLE;
    cudaSetDevice(c->device);
    c->last_launches = 0;
    if (batch == 0) return COS_OK;
    const bool two = c->table[1] && c->table[1] != c->table[0];
    const size_t one = (size_t)batch * n * n * sizeof(double);
    int rc = grow(c, (void**)&c->gscratch, &c->gscratch_bytes, two ? 2 * one : one);
    if (rc != COS_OK) return rc;
    double* gup = c->gscratch;
    double* gdn = two ? c->gscratch + (size_t)batch * n * n : gup;
    rc = do_build_G(c, n, batch, d_xy, d_tau, g_diag, gup, gdn);
    if (rc != COS_OK) return rc;
    return do_eval(c, n, batch, gup, gdn, d_u, U, d_out, 1);
}


int cos_eval_connected_xt_host(cos_ctx* c, int n, long long batch, const int* h_xy, const double* h_tau,
                               double g_diag, const double* h_u, double U, double* h_out)
{
    if (!c || n < 1 || n > COS_MAX_ORDER || batch < 0) return COS_EINVAL;
    if (batch > 0 && (!h_xy || !h_tau || !h_out)) return COS_EINVAL;
    if (!c->table[0]) return COS_ENOTABLE;
    cudaSetDevice(c->device);
    c->last_launches = 0;
    if (batch == 0) return COS_OK;
    const size_t b_xy = (size_t)batch * n * 2 * sizeof(int);
    const size_t b_tau = (size_t)batch * n * sizeof(double);
    const size_t b_u = h_u ? b_tau : 0;
    const size_t b_out = (size_t)batch * sizeof(double);
    int rc = grow(c, &c->stage, &c->stage_bytes, b_xy + b_tau + b_u + b_out);
    if (rc != COS_OK) return rc;
    char* base = (char*)c->stage;
    double* d_tau = (double*)base;
    double* d_u = h_u ? (double*)(base + b_tau) : nullptr;
    double* d_out = (double*)(base + b_tau + b_u);
    int* d_xy = (int*)(base + b_tau + b_u + b_out);
    // Two chunks when the batch is large: the host-to-device copy of the second half runs on a copy stream behind
    // the kernels of the first half.
    const int nchunk = batch >= 8192 ? 2 : 1;
    if (nchunk == 2 && !c->copy_stream) {
        COS_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (cudaEvent_t& e : c->copy_done) COS_CUDA(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    const long long b0 = nchunk == 2 ? batch / 2 : batch;
    int launches = 0;
    for (int k = 0; k < nchunk; ++k) {
        const long long lo = k == 0 ? 0 : b0, cnt = k == 0 ? b0 : batch - b0;
        cudaStream_t cs = nchunk == 2 ? c->copy_stream : c->stream;
        COS_CUDA(c, cudaMemcpyAsync(d_xy + lo * n * 2, h_xy + lo * n * 2, (size_t)cnt * n * 2 * sizeof(int), cudaMemcpyHostToDevice, cs));
        COS_CUDA(c, cudaMemcpyAsync(d_tau + lo * n, h_tau + lo * n, (size_t)cnt * n * sizeof(double), cudaMemcpyHostToDevice, cs));
        if (h_u) COS_CUDA(c, cudaMemcpyAsync(d_u + lo * n, h_u + lo * n, (size_t)cnt * n * sizeof(double), cudaMemcpyHostToDevice, cs));
        if (nchunk == 2) COS_CUDA(c, cudaEventRecord(c->copy_done[k], cs));
    }
    for (int k = 0; k < nchunk; ++k) {
        const long long lo = k == 0 ? 0 : b0, cnt = k == 0 ? b0 : batch - b0;
        if (nchunk == 2) COS_CUDA(c, cudaStreamWaitEvent(c->stream, c->copy_done[k], 0));
        rc = cos_eval_connected_xt(c, n, cnt, d_xy + lo * n * 2, d_tau + lo * n, g_diag, d_u ? d_u + lo * n : nullptr, U,
                                   d_out + lo);
        if (rc != COS_OK) return rc;
        launches += c->last_launches;
    }
    c->last_launches = launches;
    COS_CUDA(c, cudaMemcpyAsync(h_out, d_out, b_out, cudaMemcpyDeviceToHost, c->stream));
    COS_CUDA(c, cudaStreamSynchronize(c->stream));
    return COS_OK;
}

int cos_internal_device(const cos_ctx* c) { return c->device; }
void* cos_internal_stream(const cos_ctx* c) { return (void*)c->stream; }

int cos_set_loop_weight(cos_ctx* c, double n_f)
{
    if (!c || !(n_f == n_f) || n_f - n_f != 0.0) return COS_EINVAL;   // NaN / infinity
    c->loop_weight = n_f;
    return COS_OK;
}

int cos_debug_force_generic(cos_ctx* c, int enable)
{
    if (!c) return COS_EINVAL;
    c->force_generic = enable != 0;
    return COS_OK;
}

int cos_mc_run(cos_ctx* c, int n, long long walkers, int steps, unsigned long long seed, int* d_xy, double* d_tau,
               double g_diag, double U, double* d_weight, unsigned char* d_accept_hist, long long* d_accepted,
               double* d_sign_sum)
{
    if (!c || n < 1 || n > COS_MAX_ORDER || walkers < 0 || steps < 0) return COS_EINVAL;
    if (walkers > 0 && (!d_xy || !d_tau || !d_weight)) return COS_EINVAL;
    if (!c->table[0]) return COS_ENOTABLE;
    if (c->table[1] && c->table[1] != c->table[0]) return COS_EINVAL;     // one table for both species (reading R19)
    cudaSetDevice(c->device);
    c->last_launches = 0;
    if (walkers == 0) return COS_OK;
    const size_t b_xy = (size_t)walkers * n * 2 * sizeof(int), b_tau = (size_t)walkers * n * sizeof(double);
    const size_t b_w = (size_t)walkers * sizeof(double);
    int rc = grow(c, &c->mc, &c->mc_bytes, b_tau + 2 * b_w + b_xy);
    if (rc != COS_OK) return rc;
    char* base = (char*)c->mc;
    double* tau_p = (double*)base;
    double* w_new = (double*)(base + b_tau);
    double* w_alt = (double*)(base + b_tau + b_w);
    int* xy_p = (int*)(base + b_tau + 2 * b_w);
    if (d_accepted) COS_CUDA(c, cudaMemsetAsync(d_accepted, 0, (size_t)walkers * sizeof(long long), c->stream));
    if (d_sign_sum) COS_CUDA(c, cudaMemsetAsync(d_sign_sum, 0, b_w, c->stream));
    int launches = 0;
    // weight of the initial configurations; the weight of the current state then alternates between two buffers so
    // that the accept kernel never overwrites a value another thread of the same walker still has to read
    double* w_cur = (steps % 2 == 0) ? d_weight : w_alt;
    double* w_nxt = (steps % 2 == 0) ? w_alt : d_weight;
    rc = cos_eval_connected_xt(c, n, walkers, d_xy, d_tau, g_diag, nullptr, U, w_cur);
    if (rc != COS_OK) return rc;
    launches += c->last_launches;
    McArgs a{};
    a.n = n; a.walkers = walkers; a.seed = seed; a.Lx = c->Lx; a.Ly = c->Ly; a.beta = c->beta;
    a.xy = d_xy; a.tau = d_tau; a.xy_p = xy_p; a.tau_p = tau_p; a.w_new = w_new;
    a.hist = d_accept_hist; a.accepted = d_accepted; a.sign_sum = d_sign_sum;
    long long blocks = (walkers * n + 255) / 256;
    const long long cap = (long long)c->num_sms * 16;
    if (blocks > cap) blocks = cap;
    for (int step = 0; step < steps; ++step) {
        a.step = step; a.w_old = w_cur; a.w_out = w_nxt;
        mc_propose_kernel<<<(unsigned)blocks, 256, 0, c->stream>>>(a);
        COS_CUDA(c, cudaGetLastError());
        rc = cos_eval_connected_xt(c, n, walkers, xy_p, tau_p, g_diag, nullptr, U, w_new);
        if (rc != COS_OK) return rc;
        launches += c->last_launches + 2;
        mc_accept_kernel<<<(unsigned)blocks, 256, 0, c->stream>>>(a);
        COS_CUDA(c, cudaGetLastError());
        double* tmp = w_cur; w_cur = w_nxt; w_nxt = tmp;
    }
    c->last_launches = launches;      // after the last swap w_cur == d_weight
    return COS_OK;
}

int cos_last_launch_count(const cos_ctx* c) { return c ? c->last_launches : 0; }
const char* cos_last_kernel_name(const cos_ctx* c) { return c ? c->last_kernel : "none"; }

int cos_enable_kernel_timer(cos_ctx* c, int enable)
{
    if (!c) return COS_EINVAL;
    c->timing = enable != 0;
    return COS_OK;
}

int cos_reset_kernel_timer(cos_ctx* c)
{
    if (!c) return COS_EINVAL;
    c->ev_used = 0;
    return COS_OK;
}

int cos_kernel_time_ms(cos_ctx* c, double* avg_ms, long long* launches)
{
    if (!c || !avg_ms || c->ev_used == 0) return COS_EINVAL;
    cudaSetDevice(c->device);
    COS_CUDA(c, cudaStreamSynchronize(c->stream));
    double total = 0.0;
    for (size_t k = 0; k < c->ev_used; k += 2) {
        float ms = 0.f;
        COS_CUDA(c, cudaEventElapsedTime(&ms, c->ev[k], c->ev[k + 1]));
        total += ms;
    }
    *avg_ms = total / (double)(c->ev_used / 2);
    if (launches) *launches = (long long)(c->ev_used / 2);
    return COS_OK;
}

long long cos_flop_count(int n, int n_species, int connected)
{
    if (n < 1 || n > 20 || n_species < 1 || n_species > 2) return -1;
    const long long two_n = 1LL << n;
    // ext(n) = (n^2-3n+4) 2^(n-2) - 1 ; close(n) = n 2^(n-1)   (exact for n >= 1; n = 1: ext = 0)
    const long long ext = ((long long)(n * n - 3 * n + 4) * two_n) / 4 - 1;
    const long long close = (long long)n * two_n / 2;
    long long fma_total = n_species * (ext + close);
    long long flop = 2 * fma_total;
    if (connected) {
        long long p3 = 1;
        for (int i = 0; i < n - 1; ++i) p3 *= 3;
        flop += 2 * (p3 - two_n / 2);       // reduction FMAs
        flop += 2 * two_n;                   // combine: 2^n entries, counted like an FMA each
    }
    return flop;
}

}  // extern "C"
