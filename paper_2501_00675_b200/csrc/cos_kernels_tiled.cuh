// cos_kernels_tiled.cuh -- register-tiled CoS evaluation for orders whose frontier fits in shared memory.
//
// Same recursion as cos_kernels_generic.cuh with the work laid out for the FP64 pipe:
//
//  * vertices of a stage h are split into T = {0..B-1} ("thread bits") and Q = {B..h-1}.  One work item is
//    one Q-subset RQ (|RQ| = j, the "Q-level") of one configuration; the thread that owns it carries all
//    2^B subsets R = RQ + RT, RT subset of T, so every Green's function W[c][c'] it loads is used 2^B times,
//    transitions inside T never leave the register file, and every FMA executed is one the method needs
//    (no padding, no masked lanes).
//  * items of one Q-level are enumerated in colex rank order from a table built once per CTA; lanes are
//    consecutive ranks (and consecutive configurations), so the loads of node values are conflict free.
//    Node values of the 2^B subsets of an item form one padded record (RS doubles) read with LDS.128.
//  * the two loop orders "targets in registers, stream sources" (mode A) and "sources in registers, stream
//    targets" (mode B) keep the register tile at 2^B * min(#targets, #sources).
//  * several configurations share one CTA so that narrow levels still fill warps.
//
// Z[S] is kept in "rank layout": record (lvl[|SQ|] + rank(SQ)) holds Z[(SQ, ST)] for the 2^B values of ST.
#pragma once
#include "cos_common.cuh"

namespace cosb {

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

template <int B> struct Rec { static constexpr int RS = (B == 3) ? 10 : ((B == 2) ? 6 : (1 << B)); };

// Host/device sizing helpers (doubles).
template <int B>
__host__ __device__ inline int tiled_bufrec(int n)   // records in ONE level buffer (max over q, j)
{
    int best = 1;
    const int qmax = n - B;
    for (int q = 0; q < qmax; ++q)
        for (int j = 0; j <= q + 1; ++j) {
#ifdef __CUDA_ARCH__
            const int v = j * kBinom.c[q][j];
#else
            const int v = j * kBinomHost.c[q][j];
#endif
            if (v > best) best = v;
        }
    return best;
}

struct TiledDims {
    int n, G, nsp;
    int qmax;        // n - B
    int wstride;     // doubles per configuration of W (n*n rounded up to even)
    int zrec;        // records per species in Zr (2^qmax)
    int bufrec;      // records per level buffer
    int cfg_doubles; // doubles per configuration
    int tab_bytes;   // table bytes at the start of shared memory
    int use_global;  // 1: the configuration block (W, Z, level buffers, reduction arrays) lives in EvalArgs::scratch
};

template <int B>
inline TiledDims tiled_dims(int n, int G, int nsp)
{
    TiledDims d{};
    d.n = n; d.G = G; d.nsp = nsp;
    d.qmax = n - B;
    d.wstride = (n * n + 16 + 1) & ~1;                 // W + 16 slots for -u
    d.zrec = 1 << d.qmax;
    d.bufrec = tiled_bufrec<B>(n);
    const int RS = Rec<B>::RS;
    int work = 2 * d.bufrec * RS;                      // two level buffers; later D0/C' and D1
    const int need = 36 * (1 << (n - 5)) + 16;         // reduction arrays: 2 x 2^(n-5) rows x 18 doubles (cos_reduce_blocked.cuh)
    if (work < need) work = need;
    d.cfg_doubles = d.wstride + nsp * d.zrec * RS + work;
    d.cfg_doubles = (d.cfg_doubles + 1) & ~1;
    d.tab_bytes = (((2 * 2 * (1 << (n - 1)) + 4 * 64) + 15) & ~15) + 4096;   // mask16 + rank16 (2^(n-1) each) + lvlT[32] + lvlZ[32] + wtab[512]
    return d;
}

template <int B>
inline size_t tiled_smem_bytes(int n, int G, int nsp)
{
    const TiledDims d = tiled_dims<B>(n, G, nsp);
    return (size_t)d.tab_bytes + sizeof(double) * (size_t)d.cfg_doubles * G;   // all-in-shared-memory variant
}

// Everything an item routine needs that is uniform over the CTA for one level step.
struct LevelCtx {
    int n, h, q, j;          // stage vertex h = q + B, Q-level j
    int cnt, cnt_next;       // C(q, j), C(q, j+1)
    int mlvl_j;              // offset of the popcount-j list in mask16
    int lvl_j, lvl_j1;       // record offsets of Q-levels j and j+1 in Zr
    unsigned qmask;          // (1 << q) - 1
    const uint16_t* mask16;  // [lvl[j] + r] -> RQ
    const uint16_t* rank16;  // [RQ] -> colex rank within its popcount class
    int wstride, cfg_doubles;
    int off_z, off_cur, off_nxt;   // double offsets inside a configuration's block
    double* cfg0;            // configuration 0 of this CTA
};

// ---- mode A: targets in registers (N of them), sources streamed -------------------------------------
template <int B, int N>
__device__ __forceinline__ void item_mode_A(const LevelCtx& c, int g, int r)
{
    constexpr int NT = 1 << B;
    constexpr int RS = Rec<B>::RS;
    double* cfg = c.cfg0 + (size_t)g * c.cfg_doubles;
    const double* W = cfg;
    const unsigned RQ = c.mask16[c.mlvl_j + r];
    unsigned absent = ~RQ & c.qmask;
    int colb[N > 0 ? N : 1];          // vertex id of target k
    int orec[N > 0 ? N : 1];          // record index in the next level buffer
#pragma unroll
    for (int k = 0; k < N; ++k) {
        const int d = __ffs(absent) - 1;
        absent &= absent - 1;
        colb[k] = d + B;
        const unsigned R2 = RQ | (1u << d);
        orec[k] = __popc(RQ & ((1u << d) - 1)) * c.cnt_next + c.rank16[R2];
    }
    double accQ[NT][N > 0 ? N : 1], accZ[NT], accT[NT][B];
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        accZ[t] = 0.0;
#pragma unroll
        for (int k = 0; k < N; ++k) accQ[t][k] = 0.0;
#pragma unroll
        for (int tp = 0; tp < B; ++tp) accT[t][tp] = 0.0;
    }
    // phase 1: sources in Q (streamed) and the start node h
    unsigned m = RQ;
    const double* ap = cfg + c.off_cur + (size_t)r * RS;
    const int astep = c.cnt * RS;
    for (int i = 0; i <= c.j; ++i) {
        const double* rec;
        int v;
        if (i < c.j) {
            v = __ffs(m) - 1 + B;
            m &= m - 1;
            rec = ap;
            ap += astep;
        } else {
            v = c.h;
            rec = cfg + c.off_z + (size_t)(c.lvl_j + r) * RS;
        }
        const double* row = W + v * c.n;
        double a[NT];
#pragma unroll
        for (int t = 0; t < NT; t += 2) {
            const double2 x = *reinterpret_cast<const double2*>(rec + t);
            a[t] = x.x;
            a[t + 1] = x.y;
        }
#pragma unroll
        for (int k = 0; k < N; ++k) {
            const double w = row[colb[k]];
#pragma unroll
            for (int t = 0; t < NT; ++t) accQ[t][k] = fma(a[t], w, accQ[t][k]);
        }
        {
            const double w = row[c.h];
#pragma unroll
            for (int t = 0; t < NT; ++t) accZ[t] = fma(-a[t], w, accZ[t]);      // -1 per closed loop
        }
#pragma unroll
        for (int tp = 0; tp < B; ++tp) {
            const double w = row[tp];
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if (!((t >> tp) & 1)) accT[t][tp] = fma(a[t], w, accT[t][tp]);
        }
    }
    // phase 2a: transitions inside T, by |RT| (node (RT, t) = accT[RT ^ (1<<t)][t] is final when used)
#pragma unroll
    for (int l = 1; l < B; ++l)
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            if (cpopc(t) != l) continue;
#pragma unroll
            for (int ts = 0; ts < B; ++ts) {
                if (!((t >> ts) & 1)) continue;
                const double s = accT[t ^ (1 << ts)][ts];
#pragma unroll
                for (int tp = 0; tp < B; ++tp)
                    if (!((t >> tp) & 1)) accT[t][tp] = fma(s, W[ts * c.n + tp], accT[t][tp]);
            }
        }
    // phase 2b: sources in T -> targets in Q and the close
#pragma unroll
    for (int k = 0; k < N; ++k)
#pragma unroll
        for (int ts = 0; ts < B; ++ts) {
            const double w = W[ts * c.n + colb[k]];
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if ((t >> ts) & 1) accQ[t][k] = fma(accT[t ^ (1 << ts)][ts], w, accQ[t][k]);
        }
#pragma unroll
    for (int ts = 0; ts < B; ++ts) {
        const double w = W[ts * c.n + c.h];
#pragma unroll
        for (int t = 0; t < NT; ++t)
            if ((t >> ts) & 1) accZ[t] = fma(-accT[t ^ (1 << ts)][ts], w, accZ[t]);
    }
    // outputs: next-level records and Z[(RQ + {h}, RT)]
    double* nxt = cfg + c.off_nxt;
#pragma unroll
    for (int k = 0; k < N; ++k) {
        double* o = nxt + (size_t)orec[k] * RS;
#pragma unroll
        for (int t = 0; t < NT; t += 2) *reinterpret_cast<double2*>(o + t) = make_double2(accQ[t][k], accQ[t + 1][k]);
    }
    {
        const int rz = c.rank16[RQ | (1u << c.q)];
        double* o = cfg + c.off_z + (size_t)(c.lvl_j1 + rz) * RS;
#pragma unroll
        for (int t = 0; t < NT; t += 2) *reinterpret_cast<double2*>(o + t) = make_double2(accZ[t], accZ[t + 1]);
    }
}

// ---- mode B: sources in registers (J1 = j + 1 of them, the last one is h), targets streamed ----------
template <int B, int J1>
__device__ __forceinline__ void item_mode_B(const LevelCtx& c, int g, int r)
{
    constexpr int NT = 1 << B;
    constexpr int RS = Rec<B>::RS;
    double* cfg = c.cfg0 + (size_t)g * c.cfg_doubles;
    const double* W = cfg;
    const unsigned RQ = c.mask16[c.mlvl_j + r];
    double a[NT][J1];
    int rowo[J1];                     // v * n for source i
    {
        unsigned m = RQ;
        const double* ap = cfg + c.off_cur + (size_t)r * RS;
        const int astep = c.cnt * RS;
#pragma unroll
        for (int i = 0; i < J1; ++i) {
            const double* rec;
            if (i < J1 - 1) {
                rowo[i] = (__ffs(m) - 1 + B) * c.n;
                m &= m - 1;
                rec = ap;
                ap += astep;
            } else {
                rowo[i] = c.h * c.n;
                rec = cfg + c.off_z + (size_t)(c.lvl_j + r) * RS;
            }
#pragma unroll
            for (int t = 0; t < NT; t += 2) {
                const double2 x = *reinterpret_cast<const double2*>(rec + t);
                a[t][i] = x.x;
                a[t + 1][i] = x.y;
            }
        }
    }
    // nodes with current vertex in T: Q/h sources first, then inside T by |RT|
    double accT[NT][B];
#pragma unroll
    for (int t = 0; t < NT; ++t)
#pragma unroll
        for (int tp = 0; tp < B; ++tp) accT[t][tp] = 0.0;
#pragma unroll
    for (int i = 0; i < J1; ++i)
#pragma unroll
        for (int tp = 0; tp < B; ++tp) {
            const double w = W[rowo[i] + tp];
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if (!((t >> tp) & 1)) accT[t][tp] = fma(a[t][i], w, accT[t][tp]);
        }
#pragma unroll
    for (int l = 1; l < B; ++l)
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            if (cpopc(t) != l) continue;
#pragma unroll
            for (int ts = 0; ts < B; ++ts) {
                if (!((t >> ts) & 1)) continue;
                const double s = accT[t ^ (1 << ts)][ts];
#pragma unroll
                for (int tp = 0; tp < B; ++tp)
                    if (!((t >> tp) & 1)) accT[t][tp] = fma(s, W[ts * c.n + tp], accT[t][tp]);
            }
        }
    // stream the targets: absent Q vertices, then the close (column h)
    unsigned absent = ~RQ & c.qmask;
    double* nxt = cfg + c.off_nxt;
    const int ntargets = c.q - c.j;
    for (int k = 0; k <= ntargets; ++k) {
        int v;
        double* o;
        const bool is_close = (k == ntargets);
        if (!is_close) {
            const int d = __ffs(absent) - 1;
            absent &= absent - 1;
            v = d + B;
            const unsigned R2 = RQ | (1u << d);
            o = nxt + (size_t)(__popc(RQ & ((1u << d) - 1)) * c.cnt_next + c.rank16[R2]) * RS;
        } else {
            v = c.h;
            o = cfg + c.off_z + (size_t)(c.lvl_j1 + c.rank16[RQ | (1u << c.q)]) * RS;
        }
        double acc[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) acc[t] = 0.0;
#pragma unroll
        for (int i = 0; i < J1; ++i) {
            const double w = W[rowo[i] + v];
#pragma unroll
            for (int t = 0; t < NT; ++t) acc[t] = fma(a[t][i], w, acc[t]);
        }
#pragma unroll
        for (int ts = 0; ts < B; ++ts) {
            const double w = W[ts * c.n + v];
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if ((t >> ts) & 1) acc[t] = fma(accT[t ^ (1 << ts)][ts], w, acc[t]);
        }
        if (is_close) {
#pragma unroll
            for (int t = 0; t < NT; ++t) acc[t] = -acc[t];
        }
#pragma unroll
        for (int t = 0; t < NT; t += 2) *reinterpret_cast<double2*>(o + t) = make_double2(acc[t], acc[t + 1]);
    }
}

template <int B, int NA_MAX, int JB_MAX>
__device__ __forceinline__ void run_level(const LevelCtx& c, int ng, int tid, int nthreads)
{
    const int items = ng * c.cnt;
    const int N = c.q - c.j, J1 = c.j + 1;
    const bool useA = (N <= NA_MAX) && (N <= J1 || J1 > JB_MAX);
    for (int idx = tid; idx < items; idx += nthreads) {
        const int g = idx / c.cnt, r = idx - g * c.cnt;
        if (useA) {
            switch (N) {
                case 0: item_mode_A<B, 0>(c, g, r); break;
                case 1: item_mode_A<B, 1>(c, g, r); break;
                case 2: item_mode_A<B, 2>(c, g, r); break;
                case 3: item_mode_A<B, 3>(c, g, r); break;
                case 4: item_mode_A<B, 4>(c, g, r); break;
                case 5: if constexpr (NA_MAX >= 5) { item_mode_A<B, 5>(c, g, r); } break;
                default: if constexpr (NA_MAX >= 6) { item_mode_A<B, 6>(c, g, r); } break;
            }
        } else {
            switch (J1) {
                case 1: item_mode_B<B, 1>(c, g, r); break;
                case 2: item_mode_B<B, 2>(c, g, r); break;
                case 3: item_mode_B<B, 3>(c, g, r); break;
                case 4: item_mode_B<B, 4>(c, g, r); break;
                case 5: item_mode_B<B, 5>(c, g, r); break;
                case 6: if constexpr (JB_MAX >= 6) { item_mode_B<B, 6>(c, g, r); } break;
                default: if constexpr (JB_MAX >= 7) { item_mode_B<B, 7>(c, g, r); } break;
            }
        }
    }
}

// Z[RT] for RT subset of T = {0,1,2} (all stages h < B), one thread per configuration, written in the
// propagation's own order (start / extend / close), stage by stage.
template <int B>
__device__ __forceinline__ void small_stages(const double* W, int n, double* z /* record 0 of Zr */)
{
    static_assert(B == 2 || B == 3, "B");
    const double w00 = W[0], w01 = W[1], w10 = W[n], w11 = W[n + 1];
    z[0] = 1.0;
    const double z1 = -w00;                                   // stage 0
    z[1] = z1;
    const double z2 = -w11;                                   // stage 1: P[{}][1] = 1
    z[2] = z2;
    // P[{0}][1] = Z[{0}], P[{0}][0] = W[1][0]; close: Z[{0,1}] = -(P[{0}][0] W[0][1] + Z[{0}] W[1][1])
    const double z3 = -fma(w10, w01, z1 * w11);
    z[3] = z3;
    if constexpr (B == 3) {
        const double w02 = W[2], w12 = W[n + 2], w20 = W[2 * n], w21 = W[2 * n + 1], w22 = W[2 * n + 2];
        z[4] = -w22;                                          // stage 2, R = {}
        // R = {0}: nodes (R, 2) = Z[{0}] = z1, (R, 0) = W[2][0]  (from R = {} extended to 0)
        const double p0_0 = w20;                              // P[{0}][0]
        const double p1_1 = w21;                              // P[{1}][1]
        z[5] = -fma(p0_0, w02, z1 * w22);                     // Z[{0,2}]
        z[6] = -fma(p1_1, w12, z2 * w22);                     // Z[{1,2}]
        // R = {0,1}: (R,2) = Z[{0,1}] = z3; (R,1) from R={0}: P[{0}][0] W[0][1] + P[{0}][2] W[2][1];
        //            (R,0) from R={1}: P[{1}][1] W[1][0] + P[{1}][2] W[2][0]
        const double p01_1 = fma(p0_0, w01, z1 * w21);
        const double p01_0 = fma(p1_1, w10, z2 * w20);
        z[7] = -fma(p01_0, w02, fma(p01_1, w12, z3 * w22));   // Z[{0,1,2}]
    }
}

}  // namespace cosb
#include "cos_reduce_blocked.cuh"
namespace cosb {

#ifdef COS_PHASE_TIMING
__device__ unsigned long long g_phase_cycles[32];
#define COS_PHASE_MARK(k) do { __syncthreads(); if (threadIdx.x == 0) { const long long now__ = clock64(); \
    atomicAdd(&g_phase_cycles[k], (unsigned long long)(now__ - phase_t0__)); phase_t0__ = now__; } } while (0)
#else
#define COS_PHASE_MARK(k) do { } while (0)
#endif

template <int B, int THREADS, int NA_MAX, int JB_MAX, bool GLOBAL>
__global__ void __launch_bounds__(THREADS) eval_tiled_kernel(EvalArgs a, TiledDims d)
{
#ifdef COS_PHASE_TIMING
    long long phase_t0__ = clock64();
#endif
    constexpr int NT = 1 << B;
    constexpr int RS = Rec<B>::RS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint16_t* mask16 = reinterpret_cast<uint16_t*>(smem_raw);
    uint16_t* rank16 = mask16 + (1 << (d.n - 1));
    int* lvlT = reinterpret_cast<int*>(rank16 + (1 << (d.n - 1)));   // list offsets, ground set n-1 bits
    int* lvl = lvlT + 32;                                            // Zr record offsets, ground set qmax bits
    double* cfg0 = GLOBAL ? a.scratch + (size_t)blockIdx.x * a.scratch_stride
                          : reinterpret_cast<double*>(smem_raw + d.tab_bytes);
    const int tid = threadIdx.x;
    const int n = d.n, qmax = d.qmax, nsp = d.nsp;
    const unsigned N = 1u << n;

    // ---- tables: Q-subsets of {0..qmax} by popcount in colex order (rank independent of the ground set) --
    if (tid == 0) {
        int run = 0;
        for (int j = 0; j <= n; ++j) { lvlT[j] = run; run += kBinom.c[n - 1][j]; }
        run = 0;
        for (int j = 0; j <= qmax + 1; ++j) { lvl[j] = run; run += kBinom.c[qmax][j]; }
    }
    __syncthreads();
    for (unsigned mk = tid; mk < (1u << (n - 1)); mk += THREADS) {
        int rk = 0, i = 0;
        unsigned m = mk;
        while (m) { const int s = __ffs(m) - 1; m &= m - 1; ++i; rk += kBinom.c[s][i]; }
        rank16[mk] = (uint16_t)rk;
        mask16[lvlT[i] + rk] = (uint16_t)mk;
    }
    __syncthreads();

    const int off_w = 0;
    const int off_z = d.wstride;
    const int off_b0 = off_z + nsp * d.zrec * RS;
    const int off_b1 = off_b0 + d.bufrec * RS;

    const long long ngroups = (a.batch + d.G - 1) / d.G;
    for (long long grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
        const long long b0 = grp * d.G;
        const int ng = (int)min((long long)d.G, a.batch - b0);
        __syncthreads();
        COS_PHASE_MARK(0);
        for (int s = 0; s < nsp; ++s) {
            // ---- W of this species; -u_a folded into the rows of species 0 when there are two ----
            for (int t = tid; t < ng * 16; t += THREADS) {
                const int g = t >> 4, v = t & 15;
                if (v < n) cfg0[(size_t)g * d.cfg_doubles + off_w + n * n + v] = -(a.u ? a.u[(b0 + g) * n + v] : a.U);
            }
            __syncthreads();
            for (int t = tid; t < ng * n * n; t += THREADS) {
                const int g = t / (n * n), e = t - g * n * n;
                double* cfg = cfg0 + (size_t)g * d.cfg_doubles;
                const double gv = (s == 0 ? a.Gup : a.Gdn)[(b0 + g) * n * n + e];
                cfg[off_w + e] = (nsp == 2 && s == 0) ? gv * cfg[off_w + n * n + e / n] : gv;
            }
            __syncthreads();
            if (tid < ng) {
                double* cfg = cfg0 + (size_t)tid * d.cfg_doubles;
                small_stages<B>(cfg + off_w, n, cfg + off_z + (size_t)s * d.zrec * RS);
            }
            __syncthreads();
            LevelCtx c;
            c.n = n; c.mask16 = mask16; c.rank16 = rank16;
            c.wstride = d.wstride; c.cfg_doubles = d.cfg_doubles; c.cfg0 = cfg0;
            c.off_z = off_z + s * d.zrec * RS;
            for (int q = 0; q < qmax; ++q) {
                c.q = q; c.h = q + B; c.qmask = (1u << q) - 1;
                int cur = off_b0, nxt = off_b1;
                for (int j = 0; j <= q; ++j) {
                    c.j = j; c.cnt = kBinom.c[q][j]; c.cnt_next = kBinom.c[q][j + 1];
                    c.mlvl_j = lvlT[j]; c.lvl_j = lvl[j]; c.lvl_j1 = lvl[j + 1];
                    c.off_cur = cur; c.off_nxt = nxt;
                    run_level<B, NA_MAX, JB_MAX>(c, ng, tid, THREADS);
                    __syncthreads();
                    const int tmp = cur; cur = nxt; nxt = tmp;
                }
            }
        }

        COS_PHASE_MARK(1);
        // ---- a3 + a5 ("all"): D[full] ----
        const int full_rec = lvl[qmax] + 0;                  // RQ = all of Q: the only subset of size qmax
        if (!a.connected) {
            if (tid < ng) {
                double* cfg = cfg0 + (size_t)tid * d.cfg_doubles;
                const double zu = cfg[off_z + (size_t)full_rec * RS + (NT - 1)];
                const double zd = cfg[off_z + (size_t)(nsp - 1) * d.zrec * RS + (size_t)full_rec * RS + (NT - 1)];
                double w = 1.0;
                if (nsp == 1) for (int v = 0; v < n; ++v) w *= cfg[off_w + n * n + v];
                a.out[b0 + tid] = w * zu * zd;
            }
            continue;
        }

        // ---- a3: D[S] = w(S) Zup[S] Zdn[S], split by vertex 0 into D0[S'] = D[2S'+1] (becomes C' in place) and
        //      D1[U] = D[2U], both in the padded block layout of cos_reduce_blocked.cuh ----
        const int off_c = off_b0;
        const int off_d1 = off_b0 + red_rows(n) * kRowStride;
        double* wtab = reinterpret_cast<double*>(smem_raw + d.tab_bytes - 4096);   // w(S) = wtab[S & 255] * wtab[256 + (S >> 8)]
        for (int g = 0; g < ng; ++g) {
            double* cfg = cfg0 + (size_t)g * d.cfg_doubles;
            if (nsp == 1) {
                __syncthreads();
                for (int t = tid; t < 512; t += THREADS) {
                    const int vb = (t >> 8) * 8;
                    unsigned mm = (unsigned)t & 255u;
                    double w = 1.0;
                    while (mm) { const int v = vb + __ffs(mm) - 1; mm &= mm - 1; if (v < n) w *= cfg[off_w + n * n + v]; }
                    wtab[t] = w;
                }
                __syncthreads();
            }
            for (unsigned S = tid; S < N; S += THREADS) {
                const unsigned SQ = S >> B, ST = S & (NT - 1);
                const int rec = lvl[__popc(SQ)] + rank16[SQ];
                const double zu = cfg[off_z + (size_t)rec * RS + ST];
                const double zd = cfg[off_z + (size_t)(nsp - 1) * d.zrec * RS + (size_t)rec * RS + ST];
                const double w = (nsp == 1) ? wtab[S & 255u] * wtab[256u + (S >> 8)] : 1.0;
                cfg[((S & 1u) ? off_c : off_d1) + red_addr(S >> 1)] = w * zu * zd;
            }
        }
        __syncthreads();
        COS_PHASE_MARK(2);

        // ---- a4: connected reduction, a5: C'[full] ----
        reduce_blocked<THREADS>(cfg0, d.cfg_doubles, off_c, off_d1, ng, n, mask16, lvlT, tid);
        if (tid < ng) a.out[b0 + tid] = cfg0[(size_t)tid * d.cfg_doubles + off_c + red_addr((N >> 1) - 1)];
        COS_PHASE_MARK(3);
    }
}

}  // namespace cosb
