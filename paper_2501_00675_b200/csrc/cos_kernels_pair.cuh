// cos_kernels_pair.cuh -- "pair" CoS evaluation kernel (orders 5..12): the team mapping of cos_kernels_team.cuh
// with every work item split over a PAIR of adjacent lanes.
//
// What is computed is unchanged: vertices are split into T = {0,1,2} and Q = {3..n-1}; a work
// item is one Q-pattern S_Q of one propagation instance (configuration x species); all stages advance together,
// level j holds the patterns with |S_Q| = j + 1; a node record (S_Q, c) is the 8 values R_T subset of T.
//
// What changes is who holds what.  The measured limit of the team kernel was latency, not arithmetic: one
// thread carried the whole 8 x (N+1) register tile of a pattern, so a level exposed at most 35 x C threads of
// work, each with a long dependent instruction stream, and the block barrier of every level waited for it.
// Here the two lanes (2i, 2i+1) of a pair share one item and split its ROWS: lane u holds the R_T subsets
// t = 4u + r, r = 0..3 (vertex 2 absent / present):
//   * each lane loads only its half of a source record (2 x LDS.128 instead of 4) -- no duplicated traffic;
//   * both lanes read the same W entries; the shared-memory pipeline merges identical addresses of adjacent
//     lanes (measured: LDS.64 with pairwise equal addresses costs 1 cycle per warp instead of 2), so the W
//     gather costs half as many wavefronts as with one lane per item;
//   * transitions inside T' = {0,1} stay inside a lane; the 4 nodes (t, 2) that cross from lane 0 to lane 1
//     are exchanged with one round of shuffles per item;
//   * per-thread work and registers halve, the number of resident threads doubles.
// Shared-memory layout (doubles), lane fastest so that one quarter warp touches one contiguous 128-byte row:
//   record rec, chunk p in {0,1}, instance g, lane half u:   rec * 8C + p * 4C + (2g + u) * 2 + e
//   holds the value of R_T = t = 4u + 2p + e.  For C = 2 (two items per quarter warp) p is XOR-ed with the
//   parity of rec, which differs between the records two neighbouring patterns read at the same time.
//   W entry (c, c') of instance g, replica r:                (c * n + c') * 16 + r * C + g     (16 / C replicas)
#pragma once
#include "cos_common.cuh"
#include "cos_kernels_typed.cuh"   // f64::RedLayout, f64::team_reduce (connected reduction on interleaved blocks)

namespace cosb {
using namespace f64;

constexpr int kPairB = 3;            // |T|
constexpr int kPairMaxCols = 9;      // Q-targets + close held in registers (order 12: at most 8 + 1)

template <int C> struct PairLayout {
    static_assert(C == 1 || C == 2 || C == 4 || C == 8 || C == 16, "instances per team");
    static constexpr int REP = C == 1 ? 4 : 16 / C;   // W replicas: the 16 pairs of a warp read distinct banks (C = 1: 4
                                                      // replicas, some two-way conflicts, to stay inside shared memory)
    static constexpr int WE = REP * C;           // doubles per W entry
    static constexpr int CH = 4 * C;             // doubles per record chunk
    static constexpr int REC = 8 * C;            // doubles per node record
    static constexpr int SWZ = (C <= 2) ? 1 : 0; // chunk swizzle by a record-number bit (C <= 2)
    static constexpr int SWZSH = (C == 1) ? 1 : 0;   // which bit: records x, x+2 collide for C = 1, x, x+1 for C = 2
    static constexpr int PW = 16 / C;            // patterns per warp
};

// Double offset of chunk p of record rec (without the lane part).
template <int C>
__device__ __forceinline__ int pair_chunk(int rec, int p)
{
    using L = PairLayout<C>;
    return rec * L::REC + (L::SWZ ? ((p ^ (rec >> L::SWZSH)) & 1) : p) * L::CH;
}

struct PairDims {
    int n, nsp, C;
    int qmax;          // n - 3
    int pslots;        // pattern slots per pass = threads / (2C)
    int threads;
    int maxrec;        // records per frontier buffer
    int zrec;          // Z records (2^qmax)
    int ncfg;          // configuration slots of a team = C / nsp
    int red_rows;      // 2^(n-1-kRedLB) block rows of the reduction arrays
    int off_w, off_u, off_z, off_b0, off_b1;   // double offsets behind the tables
    int off_cb, off_db;                        // reduction arrays (alias the frontier buffers)
    int off_stage;                             // staging buffer: G and u of the next team (cp.async)
    int rec_doubles;                           // doubles of the record space (W gap, -u, Z, frontier / reduction)
    int tab_bytes;
    size_t smem_bytes;
};

template <int C>
inline PairDims pair_dims(int n, int nsp, int max_threads = 1024)
{
    using L = PairLayout<C>;
    PairDims d{};
    d.n = n; d.nsp = nsp; d.C = C;
    d.qmax = n - kPairB;
    int slots = team_max_patterns(n);
    slots = (slots + L::PW - 1) / L::PW * L::PW;
    if (slots * 2 * C < 64) slots = 64 / (2 * C);
    if (slots * 2 * C > max_threads) slots = max_threads / (2 * C);   // the widest levels then take two passes
    d.pslots = slots;
    d.threads = slots * 2 * C;
    int rec_even = 1, rec_odd = 1;                        // ping-pong buffers sized for the levels they hold
    for (int j = 0; j <= d.qmax; ++j) {
        const int v = j * kBinomHost.c[d.qmax][j + 1];
        if (j & 1) { if (v > rec_odd) rec_odd = v; } else { if (v > rec_even) rec_even = v; }
    }
    d.maxrec = rec_even > rec_odd ? rec_even : rec_odd;
    d.zrec = 1 << d.qmax;
    d.ncfg = C / nsp;
    d.red_rows = 1 << (n - 1 - kRedLB);
    d.off_w = 0;
    d.off_u = d.off_w + n * n * L::WE;
    d.off_z = d.off_u + (16 + 192) * d.ncfg;              // un[v][cfg] = -u_v, then the 128 + 64 products of pair_combine
    d.off_b0 = d.off_z + d.zrec * L::REC;
    d.off_b1 = d.off_b0 + rec_even * L::REC;              // level j reads buffer (j & 1), writes buffer (~j & 1)
    int work = (rec_even + rec_odd) * L::REC;
    const int need = 2 * d.red_rows * 16 * d.ncfg;
    if (work < need) work = need;
    d.off_cb = d.off_b0;
    d.off_db = d.off_b0 + d.red_rows * 16 * d.ncfg;
    d.off_stage = d.off_b0 + work;                        // staging: [C * n * n] G, [C * n] u
    d.rec_doubles = d.off_b0 + work;
    d.tab_bytes = ((2 * 2 * d.zrec + 4 * 32) + 15) & ~15;   // rank16, recSQ (ground set Q), lvlZ
    d.smem_bytes = (size_t)d.tab_bytes + sizeof(double) * (size_t)(d.off_stage + C * n * n + C * n);
    return d;
}

// Orders 14..16: Z, the frontier and the reduction arrays live in a per-CTA block of global scratch (L2 resident
// where it fits); W, the couplings, the tables and the staging buffer stay in shared memory.  Offsets are the same
// in both spaces (the W part of the scratch block is simply unused).
template <int C>
inline PairDims pair_dims_global(int n, int threads, int nsp = 1)
{
    PairDims d = pair_dims<C>(n, nsp);
    d.threads = threads;
    d.pslots = threads / (2 * C);
    d.off_stage = d.off_z;                                // shared memory: W, -u, then the staging buffer
    d.smem_bytes = (size_t)d.tab_bytes + sizeof(double) * (size_t)(d.off_stage + C * n * n + C * n);
    return d;
}

// Uniform description of one level step.
struct PairLevel {
    double lf;                  // factor of one closed loop (EvalArgs::loopf)
    int n, j;
    int cnt, cnt_next;          // patterns at levels j and j + 1
    int lvlZ_j, lvlZ_j1;        // Z record offsets of |S_Q| = j and j + 1
    int off_z, off_cur, off_nxt;
    const uint16_t* rank16;
    const uint32_t* dsc;        // item descriptors (12 words per pattern, indexed by the Z record of S_Q), global memory
};

// ---- item descriptors of the pair kernel: one 48-byte record per Q-pattern, built once per order into global
//      memory by pair_tables_kernel (the table does not fit beside the frontier in shared memory; it is read
//      through L1).  An item's prologue is three 16-byte loads instead of a chain of bit tricks and rank look-ups.
//   w0: Z record of S_Q \ {top} | h << 16 | number of Q-targets << 24
//   w1, w2: column vertices of the Q-targets (4 bits each, ascending)     w3, w4: source vertices (4 bits each)
//   w5..w11: record numbers of the Q-targets in the next level buffer (16 bits each)
constexpr int kPairDscWords = 12;

__device__ __forceinline__ int colex_rank(unsigned m)
{
    int rk = 0, i = 0;
    while (m) { const int s = __ffs(m) - 1; m &= m - 1; ++i; rk += kBinom.c[s][i]; }
    return rk;
}

__global__ void __launch_bounds__(256) pair_tables_kernel(int n, uint32_t* out)
{
    const int qmax = n - kPairB;
    for (unsigned SQ = 1 + blockIdx.x * blockDim.x + threadIdx.x; SQ < (1u << qmax); SQ += gridDim.x * blockDim.x) {
        const int j = __popc(SQ) - 1;
        const int q = 31 - __clz((int)SQ);
        const unsigned RQ = SQ ^ (1u << q);
        int lvlZ_j = 0, lvlZ_j1 = 0;
        for (int i = 0; i <= j; ++i) { if (i < j) lvlZ_j += kBinom.c[qmax][i]; lvlZ_j1 += kBinom.c[qmax][i]; }
        const int cnt_next = kBinom.c[qmax][j + 2];
        uint32_t w[kPairDscWords];
#pragma unroll
        for (int i = 0; i < kPairDscWords; ++i) w[i] = 0;
        unsigned absent = ~RQ & ((1u << q) - 1u);
        int k = 0;
        for (; absent; ++k) {
            const int d = __ffs(absent) - 1;
            absent &= absent - 1;
            const uint32_t orec = (uint32_t)(__popc(RQ & ((1u << d) - 1u)) * cnt_next + colex_rank(SQ | (1u << d)));
            w[1 + (k >> 3)] |= (uint32_t)(d + kPairB) << (4 * (k & 7));
            w[5 + (k >> 1)] |= orec << (16 * (k & 1));
        }
        w[0] = (uint32_t)(lvlZ_j + colex_rank(RQ)) | ((uint32_t)(q + kPairB) << 16) | ((uint32_t)k << 24);
        unsigned m = RQ;
        for (int i = 0; m; ++i) { const int v = __ffs(m) - 1 + kPairB; m &= m - 1; w[3 + (i >> 3)] |= (uint32_t)v << (4 * (i & 7)); }
        uint32_t* dst = out + (size_t)(lvlZ_j1 + colex_rank(SQ)) * kPairDscWords;
#pragma unroll
        for (int i = 0; i < kPairDscWords; ++i) dst[i] = w[i];
    }
}

// The 4 values (rows r = 0..3 of this lane half) of record rec.  sm already carries the lane part.
template <int C>
__device__ __forceinline__ void pair_load_rec(const double* sm, int rec, double (&a)[4])
{
    const double2 v0 = *reinterpret_cast<const double2*>(sm + pair_chunk<C>(rec, 0));
    const double2 v1 = *reinterpret_cast<const double2*>(sm + pair_chunk<C>(rec, 1));
    a[0] = v0.x; a[1] = v0.y; a[2] = v1.x; a[3] = v1.y;
}

template <int C>
__device__ __forceinline__ void pair_store_rec(double* sm, int rec, double a0, double a1, double a2, double a3)
{
    *reinterpret_cast<double2*>(sm + pair_chunk<C>(rec, 0)) = make_double2(a0, a1);
    *reinterpret_cast<double2*>(sm + pair_chunk<C>(rec, 1)) = make_double2(a2, a3);
}

// One item: Q-pattern SQ (|SQ| = j + 1, top element q, stage vertex h = q + 3) of one instance, rows 4u..4u+3.
//   sm : shared doubles, already offset by the lane part (2g + u) * 2
//   Wl : W of this instance and replica, entry (c, c') at Wl[(c * n + c') * 16]
// NC = N + 1 columns are accumulated in registers: the N = q - j Q-targets and the close (column h), together
// with the 8 T-target accumulators.  NC is the widest item of the WARP (warp-uniform, the dispatch never
// diverges); an item with fewer targets pads with dummy columns that read a valid W column and are never stored.
template <int C, int NC, int KSKIP = 0, bool LAST = true, bool DSC = false>
__device__ __forceinline__ void pair_item(const PairLevel& L, unsigned SQ, int x, int u, double* sm, const double* Wl,
                                          unsigned lanes)
{
    constexpr int kskip = KSKIP;
    constexpr bool last = LAST;
    constexpr int WE = PairLayout<C>::WE, B = kPairB, N = NC - 1;
    const int n = L.n;
    // Column window: Q-targets kskip, kskip + 1, .. of this pattern; in the LAST window of a pattern the final
    // column is the close (column h).  Patterns with more columns than the register tile holds are processed in
    // two windows (orders >= 14), each re-reading the sources.
    int colo[NC];                     // W column offset of column k
    int orec[NC];                     // record number of target k in the next buffer (-1: dummy / close)
    int zrec, h;
    unsigned long long srcs;          // source vertices, 4 bits each
    constexpr int NQ = last ? N : NC;
    if constexpr (DSC) {
        // prologue from the descriptor table (global-record variant: L1 is large there; for the shared-memory
        // variants, whose L1 is a few KB, the table reads measured slower than the bit tricks below)
        const uint4* dp = reinterpret_cast<const uint4*>(L.dsc + (size_t)(L.lvlZ_j1 + x) * kPairDscWords);
        const uint4 d0 = __ldg(dp), d1 = __ldg(dp + 1), d2 = __ldg(dp + 2);
        const uint32_t dw[kPairDscWords] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w, d2.x, d2.y, d2.z, d2.w};
        zrec = (int)(dw[0] & 0xffffu);
        h = (int)((dw[0] >> 16) & 15u);
        const int nown = (int)(dw[0] >> 24);
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            const int t = kskip + k;                       // target index (compile time after unrolling)
            if (k < NQ && t < nown) {
                colo[k] = (int)((dw[1 + (t >> 3)] >> (4 * (t & 7))) & 15u) * WE;
                orec[k] = (int)((dw[5 + (t >> 1)] >> (16 * (t & 1))) & 0xffffu);
            } else {
                colo[k] = h * WE;      // dummy column, or the close
                orec[k] = -1;
            }
        }
        srcs = (unsigned long long)dw[3] | ((unsigned long long)dw[4] << 32);
    } else {
        const int q = 31 - __clz((int)SQ);
        const unsigned RQ = SQ ^ (1u << q);
        h = q + B;
        zrec = L.lvlZ_j + L.rank16[RQ];
        unsigned absent = ~RQ & ((1u << q) - 1u);
        for (int i = 0; i < kskip; ++i) absent &= absent - 1;
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            if (k < NQ && absent) {
                const int d = __ffs(absent) - 1;
                absent &= absent - 1;
                colo[k] = (d + B) * WE;
                orec[k] = __popc(RQ & ((1u << d) - 1u)) * L.cnt_next + L.rank16[SQ | (1u << d)];
            } else {
                colo[k] = h * WE;      // dummy column, or the close
                orec[k] = -1;
            }
        }
        srcs = RQ;                     // the loop below peels the source vertices off this mask
    }
    const int rowstride = n * WE;
    double acc[4][NC];
    double T00, T01, T11, T20, T02, T12, T22, T32;     // T_{r,tp}: node (R_T = t + {tp}, tp), t = 4u + r
    // ---- the start node (S, h) = Z[S \ {h}] ("top node", one per stage) ----
    {
        double a[4];
        pair_load_rec<C>(sm + L.off_z, zrec, a);
        const double* row = Wl + h * rowstride;
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            const double w = row[colo[k]];
#pragma unroll
            for (int r = 0; r < 4; ++r) acc[r][k] = a[r] * w;
        }
        const double w0 = row[0], w1 = row[WE], w2 = row[2 * WE];
        T00 = a[0] * w0; T20 = a[2] * w0;
        T01 = a[0] * w1; T11 = a[1] * w1;
        T02 = a[0] * w2; T12 = a[1] * w2; T22 = a[2] * w2; T32 = a[3] * w2;
    }
    // ---- sources in Q, streamed from the level buffer ----
    {
        int rec = x;
        for (int i = 0; i < L.j; ++i) {
            int v;
            if constexpr (DSC) { v = (int)(srcs & 15u); srcs >>= 4; }
            else { const unsigned mm = (unsigned)srcs; v = __ffs(mm) - 1 + B; srcs = mm & (mm - 1); }
            double a[4];
            pair_load_rec<C>(sm + L.off_cur, rec, a);
            rec += L.cnt;
            const double* row = Wl + v * rowstride;
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                const double w = row[colo[k]];
#pragma unroll
                for (int r = 0; r < 4; ++r) acc[r][k] = fma(a[r], w, acc[r][k]);
            }
            const double w0 = row[0], w1 = row[WE], w2 = row[2 * WE];
            T00 = fma(a[0], w0, T00); T20 = fma(a[2], w0, T20);
            T01 = fma(a[0], w1, T01); T11 = fma(a[1], w1, T11);
            T02 = fma(a[0], w2, T02); T12 = fma(a[1], w2, T12); T22 = fma(a[2], w2, T22); T32 = fma(a[3], w2, T32);
        }
    }
    // ---- transitions inside T.  Lane 0 (vertex 2 absent) first completes its nodes (t, 2); they are the nodes
    //      (4 + r, 2) of lane 1, which receives them by shuffle and then completes its own T' = {0,1} nodes. ----
    const double W01 = Wl[(0 * n + 1) * WE], W02 = Wl[(0 * n + 2) * WE];
    const double W10 = Wl[(1 * n + 0) * WE], W12 = Wl[(1 * n + 2) * WE];
    const double W20 = Wl[(2 * n + 0) * WE], W21 = Wl[(2 * n + 1) * WE];
    if (u == 0) {
        T11 = fma(T00, W01, T11); T20 = fma(T01, W10, T20);
        T12 = fma(T00, W02, T12); T22 = fma(T01, W12, T22);
        T32 = fma(T20, W02, fma(T11, W12, T32));
    }
    double X0 = __shfl_xor_sync(lanes, T02, 1), X1 = __shfl_xor_sync(lanes, T12, 1);
    double X2 = __shfl_xor_sync(lanes, T22, 1), X3 = __shfl_xor_sync(lanes, T32, 1);
    if (u == 0) {
        X0 = 0.0; X1 = 0.0; X2 = 0.0; X3 = 0.0;
    } else {
        T00 = fma(X0, W20, T00); T01 = fma(X0, W21, T01);
        T11 = fma(X1, W21, T11); T20 = fma(X2, W20, T20);
        T11 = fma(T00, W01, T11); T20 = fma(T01, W10, T20);
    }
    // ---- sources in T -> Q-targets and the close ----
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const double w0 = Wl[colo[k]], w1 = Wl[rowstride + colo[k]], w2 = Wl[2 * rowstride + colo[k]];
        acc[0][k] = fma(X0, w2, acc[0][k]);
        acc[1][k] = fma(X1, w2, fma(T00, w0, acc[1][k]));
        acc[2][k] = fma(X2, w2, fma(T01, w1, acc[2][k]));
        acc[3][k] = fma(X3, w2, fma(T20, w0, fma(T11, w1, acc[3][k])));
    }
    // ---- outputs: next-level records, and Z[(SQ, R_T)] = -close (one -1 per closed fermion loop) ----
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        if (orec[k] < 0) continue;
        pair_store_rec<C>(sm + L.off_nxt, orec[k], acc[0][k], acc[1][k], acc[2][k], acc[3][k]);
    }
    if (last) pair_store_rec<C>(sm + L.off_z, L.lvlZ_j1 + x, L.lf * acc[0][N], L.lf * acc[1][N], L.lf * acc[2][N], L.lf * acc[3][N]);
}

template <int C, int NCMAX, int KSKIP, bool DSC>
__device__ __forceinline__ void pair_item_switch(int ncols, const PairLevel& L, unsigned SQ, int x, int u, double* sm,
                                                 const double* Wl, unsigned lanes)
{
#define COS_PAIR_CASE(K) case K: if (K <= NCMAX) { pair_item<C, (K <= NCMAX ? K : 1), KSKIP, true, DSC>(L, SQ, x, u, sm, Wl, lanes); break; }
    switch (ncols) {
        COS_PAIR_CASE(1) COS_PAIR_CASE(2) COS_PAIR_CASE(3) COS_PAIR_CASE(4) COS_PAIR_CASE(5)
        COS_PAIR_CASE(6) COS_PAIR_CASE(7) COS_PAIR_CASE(8) COS_PAIR_CASE(9)
        default: pair_item<C, NCMAX, KSKIP, true, DSC>(L, SQ, x, u, sm, Wl, lanes); break;
    }
#undef COS_PAIR_CASE
}

// WINDOWS: patterns may have more columns than MAXNC (orders >= 14) and are then processed in two column windows.
template <int C, int MAXNC, bool WINDOWS>
__device__ __forceinline__ void pair_dispatch_item(const PairLevel& L, unsigned SQ, int x, int u, double* sm,
                                                   const double* Wl, bool active)
{
    // warp-uniform column count: the widest item of the warp (all 32 lanes call this)
    const int Nown = active ? (31 - __clz((int)SQ)) - L.j : 0;
    const int N = __reduce_max_sync(0xffffffffu, Nown);
    // both lanes of a pair are active together, so the shuffles inside an item see their partner
    const unsigned lanes = __ballot_sync(0xffffffffu, active);
    if (!active) return;
    if (!WINDOWS || N + 1 <= MAXNC) {
        pair_item_switch<C, MAXNC, 0, WINDOWS>(N + 1, L, SQ, x, u, sm, Wl, lanes);
    } else if constexpr (WINDOWS) {            // MAXNC Q-targets, then the rest and the close
        pair_item<C, MAXNC, 0, false, true>(L, SQ, x, u, sm, Wl, lanes);
        pair_item_switch<C, MAXNC, MAXNC, true>(N + 1 - MAXNC, L, SQ, x, u, sm, Wl, lanes);
    }
}

// Z[(SQ = {}, R_T)] for the 8 subsets of T (stages h < 3), one thread per instance, in the propagation's own
// order (start / extend / close).  Wl: W of this instance (any replica); zr: Z record 0 + 4g doubles.
template <int C>
__device__ __forceinline__ void pair_small_stages(const double* Wl, int n, double* zr, double lf)
{
    constexpr int WE = PairLayout<C>::WE;
    auto W = [&](int a, int b) { return Wl[(a * n + b) * WE]; };
    const double w00 = W(0, 0), w01 = W(0, 1), w02 = W(0, 2);
    const double w10 = W(1, 0), w11 = W(1, 1), w12 = W(1, 2);
    const double w20 = W(2, 0), w21 = W(2, 1), w22 = W(2, 2);
    double z[8];
    z[0] = 1.0;                                           // top node
    z[1] = lf * w00;                                      // stage 0 (lf: factor of one closed loop)
    z[2] = lf * w11;                                      // stage 1, R = {}
    z[3] = lf * fma(w10, w01, z[1] * w11);                // stage 1, R = {0}: nodes (R,0) = W[1][0], (R,1) = Z[{0}]
    z[4] = lf * w22;                                      // stage 2, R = {}
    z[5] = lf * fma(w20, w02, z[1] * w22);                // R = {0}
    z[6] = lf * fma(w21, w12, z[2] * w22);                // R = {1}
    const double p01_1 = fma(w20, w01, z[1] * w21);       // node ({0,1}, 1) from R = {0}
    const double p01_0 = fma(w21, w10, z[2] * w20);       // node ({0,1}, 0) from R = {1}
    z[7] = lf * fma(p01_0, w02, fma(p01_1, w12, z[3] * w22)); // R = {0,1}
#pragma unroll
    for (int uu = 0; uu < 2; ++uu)
#pragma unroll
        for (int p = 0; p < 2; ++p)                       // record 0: chunk p, value t = 4u + 2p + e
            *reinterpret_cast<double2*>(zr + pair_chunk<C>(0, p) + uu * 2) = make_double2(z[4 * uu + 2 * p], z[4 * uu + 2 * p + 1]);
}

// a3: D[S] = w(S) Zup[S] Zdn[S] for the NC configurations of the team, written straight into the reduction
// arrays: S odd -> CB (D0[S >> 1]), S even -> DB (D1[S >> 1]).  One thread per (Z record, configuration): the 8
// values R_T of record S_Q are the lo-values (S_Q & 3) * 4 + {0..3} of row hi = S_Q >> 2 in both arrays.
// un[v * NC + cg] = -u_v of configuration cg (aliased species only; otherwise -u is folded into W).
template <int C, int NC>
__device__ __forceinline__ void pair_combine(double* smd, double* rb, const PairDims& d, int ncfg,
                                             const uint16_t* recSQ, int tid, int nthreads)
{
    using R = RedLayout<NC>;
    constexpr int NSP = C / NC;
    double* CB = rb + d.off_cb;
    double* DB = rb + d.off_db;
    const double* un = smd + d.off_u;
    const int cg = tid % NC;
    // w(S_Q) = wt[S_Q & 127] * wt[128 + (S_Q >> 7)]: products over the 7 low / 6 high vertices of Q, once per team
    double* wt = smd + d.off_u + 16 * NC;
    if (NSP == 1) {
        for (int t = tid / NC; t < 192; t += nthreads / NC) {
            unsigned m = t < 128 ? (unsigned)t : (unsigned)(t - 128) << 7;
            double w = 1.0;
            while (m) { const int v = __ffs(m) - 1; m &= m - 1; if (v < d.qmax) w *= un[(v + kPairB) * NC + cg]; }
            wt[t * NC + cg] = w;
        }
        __syncthreads();
    }
    if (cg >= ncfg) return;
    double wT[8];
#pragma unroll
    for (int t = 0; t < 8; ++t) wT[t] = 1.0;
    if (NSP == 1) {
        const double u0 = un[0 * NC + cg], u1 = un[1 * NC + cg], u2 = un[2 * NC + cg];
#pragma unroll
        for (int t = 0; t < 8; ++t) wT[t] = ((t & 1) ? u0 : 1.0) * ((t & 2) ? u1 : 1.0) * ((t & 4) ? u2 : 1.0);
    }
    for (int rec = tid / NC; rec < d.zrec; rec += nthreads / NC) {
        const unsigned SQ = recSQ[rec];
        const double wq = (NSP == 1) ? wt[(SQ & 127u) * NC + cg] * wt[(128u + (SQ >> 7)) * NC + cg] : 1.0;
        const double* zup = rb + d.off_z + (cg * NSP) * 4;
        const double* zdn = rb + d.off_z + (cg * NSP + NSP - 1) * 4;
        double val[8];
#pragma unroll
        for (int pi = 0; pi < 4; ++pi) {                  // values t = 2 pi, 2 pi + 1: lane half pi >> 1, chunk pi & 1
            const int o = pair_chunk<C>(rec, pi & 1) + (pi >> 1) * 2;
            const double2 zu = *reinterpret_cast<const double2*>(zup + o);
            const double2 zd = *reinterpret_cast<const double2*>(zdn + o);
            val[2 * pi] = (wq * wT[2 * pi]) * (zu.x * zd.x);
            val[2 * pi + 1] = (wq * wT[2 * pi + 1]) * (zu.y * zd.y);
        }
        const unsigned hi = SQ >> 2;
        const int pa = (int)(SQ & 3u) * 2, sw = red_swz<NC>(hi);
        double* crow = CB + (int)hi * R::ROW + cg * 2;
        double* drow = DB + (int)hi * R::ROW + cg * 2;
        *reinterpret_cast<double2*>(crow + ((pa) ^ sw) * R::PSTR) = make_double2(val[1], val[3]);
        *reinterpret_cast<double2*>(crow + ((pa + 1) ^ sw) * R::PSTR) = make_double2(val[5], val[7]);
        *reinterpret_cast<double2*>(drow + ((pa) ^ sw) * R::PSTR) = make_double2(val[0], val[2]);
        *reinterpret_cast<double2*>(drow + ((pa + 1) ^ sw) * R::PSTR) = make_double2(val[4], val[6]);
    }
}

template <int C, int MAXT, int MINB, int MAXNC, bool GLOBAL = false>
__global__ void __launch_bounds__(MAXT, MINB) eval_pair_kernel(EvalArgs a, PairDims d)
{
    using Lay = PairLayout<C>;
    constexpr int WE = Lay::WE, REP = Lay::REP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
#ifdef COS_PHASE_TIMING
    long long phase_t0__ = clock64();
#endif
    // subsets of Q by popcount in colex order (rank independent of the ground set): rank16[mask], recSQ[lvlZ[|S|] + rank]
    uint16_t* rank16 = reinterpret_cast<uint16_t*>(smem_raw);
    uint16_t* recSQ = rank16 + (1 << d.qmax);                        // Z record -> S_Q (also the reduction's row lists)
    int* lvlZ = reinterpret_cast<int*>(recSQ + (1 << d.qmax));       // Z record offsets, ground set qmax bits
    const uint16_t* mask16 = recSQ;
    const int* lvlT = lvlZ;
    double* smd = reinterpret_cast<double*>(smem_raw + d.tab_bytes);
    double* rb = GLOBAL ? a.scratch + (size_t)blockIdx.x * a.scratch_stride : smd;   // record space
    const int tid = threadIdx.x, nthreads = blockDim.x;
    const int n = d.n, qmax = d.qmax, nsp = d.nsp;
    const unsigned NS = 1u << n;
    const int u = tid & 1;                       // lane half: vertex 2 absent / present in this lane's rows
    const int g = (tid >> 1) % C;                // instance of this thread
    const int slot = tid / (2 * C);              // pattern slot
    const int rep = slot % REP;                  // W replica read by this thread
    double* sm = rb + (2 * g + u) * 2;
    const double* Wl = smd + d.off_w + rep * C + g;

    // the first team's inputs are fetched while the tables are being built
    double* stage = smd + d.off_stage;
    {
        const long long total_inst0 = a.batch * nsp;
        const long long nx0 = (long long)blockIdx.x * C;
        if (nx0 < total_inst0)
            team_prefetch_inputs<C>(a, n, nsp, stage, nx0, (int)min((long long)C, total_inst0 - nx0), tid, nthreads);
    }
    if (tid == 0) {
        int run = 0;
        for (int j = 0; j <= qmax + 1; ++j) { lvlZ[j] = run; run += kBinom.c[qmax][j]; }
    }
    __syncthreads();
    for (unsigned mk = tid; mk < (1u << qmax); mk += nthreads) {
        int rk = 0, i = 0;
        unsigned m = mk;
        while (m) { const int s = __ffs(m) - 1; m &= m - 1; ++i; rk += kBinom.c[s][i]; }
        rank16[mk] = (uint16_t)rk;
        recSQ[lvlZ[i] + rk] = (uint16_t)mk;
    }
    __syncthreads();

    const long long total_inst = a.batch * nsp;
    const long long nteams = (total_inst + C - 1) / C;
    for (long long team = blockIdx.x; team < nteams; team += gridDim.x) {
        const long long inst0 = team * C;
        const int ninst = (int)min((long long)C, total_inst - inst0);
        const int ncfg = ninst / nsp;
        const long long cfgbase = inst0 / nsp;
        cp_async_wait_all();
        __syncthreads();
        team_unpack_inputs<C, REP>(a, n, nsp, stage, smd + d.off_w, smd + d.off_u, ninst, tid, nthreads);
        __syncthreads();
        if (team + gridDim.x < nteams) {
            const long long nx0 = (team + gridDim.x) * C;
            team_prefetch_inputs<C>(a, n, nsp, stage, nx0, (int)min((long long)C, total_inst - nx0), tid, nthreads);
        }
        COS_PHASE_MARK(0);
        if (tid < ninst) pair_small_stages<C>(smd + d.off_w + tid, n, rb + d.off_z + tid * 4, a.loopf);
        __syncthreads();
        COS_PHASE_MARK(1);

        // ---- a2: all stages together, level j = |S_Q| - 1; level j reads buffer (j & 1) and writes the other ----
        PairLevel L;
        L.n = n; L.rank16 = rank16; L.off_z = d.off_z; L.lf = a.loopf; L.dsc = reinterpret_cast<const uint32_t*>(a.tabs);
        for (int j = 0; j < qmax; ++j) {
            L.j = j;
            L.cnt = kBinom.c[qmax][j + 1];
            L.cnt_next = kBinom.c[qmax][j + 2];
            L.lvlZ_j = lvlZ[j]; L.lvlZ_j1 = lvlZ[j + 1];
            L.off_cur = (j & 1) ? d.off_b1 : d.off_b0;
            L.off_nxt = (j & 1) ? d.off_b0 : d.off_b1;
            const uint16_t* masks = mask16 + lvlT[j + 1];
            for (int x0 = 0; x0 < L.cnt; x0 += d.pslots) {
                const int x = x0 + slot;
                const bool active = (x < L.cnt) && (g < ninst);
                pair_dispatch_item<C, MAXNC, GLOBAL>(L, active ? masks[x] : 1u, x, u, sm, Wl, active);
            }
            __syncthreads();
            COS_PHASE_MARK(2 + j);
        }

        // ---- a3 + a5 ("all"): D[full] = w * Zup[full] * Zdn[full]; S_Q = Q, R_T = T: lane half 1, chunk 1, e = 1 ----
        if (!a.connected) {
            if (tid < ncfg) {
                const double* zp = rb + d.off_z + pair_chunk<C>(lvlZ[qmax], 1) + 2 + 1;
                const double zu = zp[(tid * nsp) * 4];
                const double zd = zp[(tid * nsp + nsp - 1) * 4];
                double w = 1.0;
                if (nsp == 1) for (int v = 0; v < n; ++v) w *= smd[d.off_u + v * C + tid];
                a.out[cfgbase + tid] = w * zu * zd;
            }
            continue;
        }

        // ---- a3: combine, a4: connected reduction, a5: C'[full] ----
        double* CB = rb + d.off_cb;
        double* DB = rb + d.off_db;
        if (nsp == 1) {
            pair_combine<C, C>(smd, rb, d, ncfg, recSQ, tid, nthreads);
            __syncthreads();
            COS_PHASE_MARK(12);
            team_reduce<C>(CB, DB, ncfg, n, mask16, lvlT, tid, nthreads);
            COS_PHASE_MARK(13);
            if (tid < ncfg) a.out[cfgbase + tid] = CB[red_elem<C>((NS >> (1 + kRedLB)) - 1, 15u, tid)];
        } else if constexpr (C >= 2) {
            pair_combine<C, C / 2>(smd, rb, d, ncfg, recSQ, tid, nthreads);
            __syncthreads();
            COS_PHASE_MARK(12);
            team_reduce<C / 2>(CB, DB, ncfg, n, mask16, lvlT, tid, nthreads);
            COS_PHASE_MARK(13);
            if (tid < ncfg) a.out[cfgbase + tid] = CB[red_elem<C / 2>((NS >> (1 + kRedLB)) - 1, 15u, tid)];
        }
    }
}

}  // namespace cosb
