// cos_kernels_team.cuh -- "team" CoS evaluation kernel: the fast path for orders whose working set of
// C propagation instances fits in the shared memory of one SM.
//
// The recursion is the one of cos_kernels_generic.cuh; what changes is the mapping:
//
//  * a "propagation instance" is one (configuration, species) pair, i.e. one n x n matrix W.  A CTA works on
//    a TEAM of C instances at a time; the lanes of a warp are  C instances x (32 / C) subset patterns, instance
//    fastest.  Every shared-memory structure is instance-interleaved, so the lanes of one wavefront
//    (quarter warp for LDS.128, half warp for LDS.64) touch one contiguous 128-byte row:
//        node record (S_Q, c)   : [part 0..3][instance 0..C-1][2 doubles]   (the 8 values R_T subset of T)
//        W entry (c, c')        : [replica 0..REP-1][instance 0..C-1]        REP = 16 / C  (C < 16)
//    The W gather is the only lane-dependent address; with REP replicas the (at most 16 / C) patterns of a
//    half warp read different bank groups, so it is conflict free by construction.  For C = 4 a quarter warp
//    spans two patterns; the part index of a record is XOR-ed with the parity of the record number so that
//    consecutive records (consecutive patterns read the same source position) use different halves of a
//    128-byte row.
//  * vertices are split into T = {0,1,2} and Q = {3..n-1} as in the tiled kernel: one thread carries the 8
//    subsets R_T of one Q-pattern, every W entry it loads is used 8 times, transitions inside T stay in
//    registers, and every FMA executed is one the method needs.
//  * ALL stages h advance together: level j holds every node (S, c) whose Q-part S_Q has j + 1 elements
//    (its top element is the stage vertex h).  Patterns of one level are the (j+1)-subsets of Q in colex
//    order -- which sorts by h first -- so there are only n - 3 block barriers per propagation instead of
//    (n-3)(n-2)/2, and a level exposes C(n-3, j+1) x C items of parallel work.
//  * the two species of one configuration are two instances of the same team, so G_up != G_dn costs no
//    extra shared memory per instance.
//  * the connected reduction (step a4) runs on configuration-interleaved blocks of 16 values (the 4 lowest
//    vertices of S' in registers), the terms of one output split over up to 32 / NC lanes of one warp.
#pragma once
#include "cos_common.cuh"
#include "cos_kernels_generic.cuh"

namespace cosb {

constexpr int kTeamB = 3;          // |T|
constexpr int kTeamNT = 8;         // 2^|T|
constexpr int kTeamMaxTargets = 6; // Q-targets held in registers (orders <= 10 need at most 6)
constexpr int kRedLB = 4;          // low bits of S' held in registers by the reduction

template <int C> struct TeamLayout {
    static_assert(C == 4 || C == 8 || C == 16 || C == 32, "instances per team");
    static constexpr int REP = (C >= 16) ? 1 : 16 / C;   // W replicas
    static constexpr int WE = REP * C;                   // doubles per W entry
    static constexpr int PART = 2 * C;                   // doubles per record part
    static constexpr int REC = 8 * C;                    // doubles per node record
    static constexpr int SWZ = (C >= 8) ? 0 : (8 / C - 1);   // part-index swizzle mask (by record number)
};

// Pointers to the even (0, 2) and odd (1, 3) parts of record `rec`: part p lives at (p & 1 ? odd : even) + p * PART.
template <int C>
struct RecPtr {
    double* even;
    double* odd;
    __device__ __forceinline__ RecPtr(double* base, int rec)
    {
        using L = TeamLayout<C>;
        double* p = base + rec * L::REC;
        if (L::SWZ) {
            const int b = (rec & 1) * L::PART;
            even = p + b;
            odd = p - b;
        } else {
            even = odd = p;
        }
    }
    __device__ __forceinline__ double* part(int p) const { return ((p & 1) ? odd : even) + p * TeamLayout<C>::PART; }
};

struct TeamDims {
    int n, nsp, C;
    int qmax;          // n - 3
    int pslots;        // pattern slots per pass = threads / C
    int threads;
    int maxrec;        // records per frontier buffer
    int zrec;          // Z records (2^qmax)
    int ncfg;          // configurations per team = C / nsp
    int red_rows;      // 2^(n-1-kRedLB) block rows of the reduction arrays
    int off_w, off_u, off_z, off_b0, off_b1;   // double offsets behind the tables
    int off_cb, off_db;                        // reduction arrays (alias the frontier buffers)
    int off_stage;                             // staging buffer: u of the next team (cp.async)
    int dsc_off;                               // byte offset of the item descriptors inside the table area
    int tab_bytes;
    size_t smem_bytes;
};

inline int team_max_patterns(int n)
{
    const int qmax = n - kTeamB;
    int best = 1;
    for (int j = 0; j < qmax; ++j) if (kBinomHost.c[qmax][j + 1] > best) best = kBinomHost.c[qmax][j + 1];
    return best;
}

template <int C>
inline TeamDims team_dims(int n, int nsp)
{
    using L = TeamLayout<C>;
    TeamDims d{};
    d.n = n; d.nsp = nsp; d.C = C;
    d.qmax = n - kTeamB;
    const int lanes_pat = 32 / C;                         // patterns per warp
    int slots = team_max_patterns(n);
    slots = (slots + lanes_pat - 1) / lanes_pat * lanes_pat;
    if (slots * C < 64) slots = 64 / C;
    d.pslots = slots;
    d.threads = slots * C;
    int maxrec = 1;
    for (int j = 0; j <= d.qmax; ++j) {
        const int v = j * kBinomHost.c[d.qmax][j + 1];
        if (v > maxrec) maxrec = v;
    }
    d.maxrec = maxrec;
    d.zrec = 1 << d.qmax;
    d.ncfg = C / nsp;
    d.red_rows = 1 << (n - 1 - kRedLB);
    d.off_w = 0;
    d.off_u = d.off_w + n * n * L::WE;
    d.off_z = d.off_u + 40 * d.ncfg;                      // un[v][cfg] = -u_v, then the 16 + 8 products of team_combine
    d.off_b0 = d.off_z + d.zrec * L::REC;
    int work = 2 * maxrec * L::REC;
    const int need = 2 * d.red_rows * 16 * d.ncfg;
    if (work < need) work = need;
    d.off_b1 = d.off_b0 + maxrec * L::REC;
    d.off_cb = d.off_b0;
    d.off_db = d.off_b0 + d.red_rows * 16 * d.ncfg;
    d.off_stage = d.off_b0 + work;                        // staging: [C * n] u of the next team
    d.dsc_off = ((2 * 2 * (1 << (n - 1)) + 4 * 64 + 2 * d.zrec) + 31) & ~31;     // mask16, rank16, lvlT, lvlZ, recSQ
    d.tab_bytes = d.dsc_off + 32 * d.zrec + 512;                                  // + one 32-byte descriptor per pattern + column units of levels 0, 1
    d.smem_bytes = (size_t)d.tab_bytes + sizeof(double) * (size_t)(d.off_stage + C * n);
    return d;
}

// Uniform description of one level step.
struct TeamLevel {
    double lf;                  // factor of one closed loop (EvalArgs::loopf)
    int n, j;
    int cnt, cnt_next;          // patterns at levels j and j + 1
    int lvlZ_j, lvlZ_j1;        // Z record offsets of |S_Q| = j and j + 1
    int off_z, off_cur, off_nxt;
    const uint16_t* rank16;
};

template <int C>
__device__ __forceinline__ void team_load_rec(const RecPtr<C>& r, double (&a)[kTeamNT])
{
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const double2 v2 = *reinterpret_cast<const double2*>(r.part(p));
        a[2 * p] = v2.x;
        a[2 * p + 1] = v2.y;
    }
}

// One item: Q-pattern SQ (|SQ| = j + 1, top element q, stage vertex h = q + 3) of one instance.
//   sm : shared doubles, already offset by the instance (g * 2)
//   Wl : W of this instance and replica, entry (c, c') at Wl[(c * n + c') * WE]
// N = q - j Q-targets are accumulated in registers together with the close (column h) and the T-targets.
// N is the number of Q-targets of the widest item of the WARP (warp-uniform, so the dispatch never diverges); an
// item with fewer targets (Nown < N) pads with dummy targets that read a valid W column and are never stored.
// Item descriptor of pattern S_Q (8 words, indexed by the Z record number of S_Q), built once per CTA: everything
// an item needs to know about the graph, so that its prologue is one wide load instead of a chain of bit tricks
// and rank look-ups (the measured critical path of a level was that chain, not the arithmetic).
//   w0: S_Q | Z record of S_Q \ {top} << 16        w1..w3: record numbers of the (at most 6) Q-targets, 16 bits each
//   w4: column vertices of the Q-targets, 4 bits each (padding: h); bits 24..27: h; bits 28..31: number of Q-targets
//   w5: source vertices (elements of S_Q \ {top}, ascending, + 3), 4 bits each
__device__ __forceinline__ void team_build_descriptor(uint32_t* dsc, unsigned SQ, int qmax, const int* lvlZ,
                                                      const uint16_t* rank16)
{
    constexpr int B = kTeamB;
    const int j = __popc(SQ) - 1;
    const int q = 31 - __clz((int)SQ);
    const unsigned RQ = SQ ^ (1u << q);
    const int h = q + B;
    const int cnt_next = kBinom.c[qmax][j + 2];
    uint32_t w[8] = {0, 0xffffffffu, 0xffffffffu, 0xffffffffu, 0, 0, 0, 0};
    w[0] = SQ | ((uint32_t)(lvlZ[j] + rank16[RQ]) << 16);
    unsigned absent = ~RQ & ((1u << q) - 1u);
    int k = 0;
    uint32_t cols = 0;
    for (; absent && k < kTeamMaxTargets; ++k) {
        const int dd = __ffs(absent) - 1;
        absent &= absent - 1;
        const uint32_t orec = (uint32_t)(__popc(RQ & ((1u << dd) - 1u)) * cnt_next + rank16[SQ | (1u << dd)]);
        const int wi = 1 + (k >> 1), sh = (k & 1) * 16;
        w[wi] = (w[wi] & ~(0xffffu << sh)) | (orec << sh);
        cols |= (uint32_t)(dd + B) << (4 * k);
    }
    const int nown = k;
    for (; k < kTeamMaxTargets; ++k) cols |= (uint32_t)h << (4 * k);
    w[4] = cols | ((uint32_t)h << 24) | ((uint32_t)nown << 28);
    unsigned m = RQ;
    for (int i = 0; m; ++i) { const int v = __ffs(m) - 1 + B; m &= m - 1; w[5] |= (uint32_t)v << (4 * i); }
#pragma unroll
    for (int i = 0; i < 8; ++i) dsc[i] = w[i];
}

template <int C, int N>
__device__ __forceinline__ void team_item(const TeamLevel& L, const uint32_t* dsc, int x, double* sm, const double* Wl)
{
    using Lay = TeamLayout<C>;
    constexpr int WE = Lay::WE, NT = kTeamNT, B = kTeamB;
    const int n = L.n;
    const uint4 d0 = *reinterpret_cast<const uint4*>(dsc);
    const uint2 d1 = *reinterpret_cast<const uint2*>(dsc + 4);
    const int zrec = (int)(d0.x >> 16);
    const int h = (int)((d1.x >> 24) & 15u);
    int colo[N + 1];                  // W column offset of target k; the last one is the close column h
    int orec[N > 0 ? N : 1];          // record number of target k in the next buffer (0xffff: dummy target)
#pragma unroll
    for (int k = 0; k < N; ++k) {
        colo[k] = (int)((d1.x >> (4 * k)) & 15u) * WE;
        const uint32_t pr = (k >> 1) == 0 ? d0.y : ((k >> 1) == 1 ? d0.z : d0.w);
        orec[k] = (int)((k & 1) ? (pr >> 16) : (pr & 0xffffu));
    }
    colo[N] = h * WE;
    unsigned srcs = d1.y;
    const int rowstride = n * WE;
    double acc[NT][N + 1], accT[NT][B];
    // ---- phase 1a: the start node (S, h) = Z[S \ {h}] ("top node", one per stage) ----
    {
        const RecPtr<C> zp(sm + L.off_z, zrec);
        double a[NT];
        team_load_rec<C>(zp, a);
        const double* row = Wl + h * rowstride;
#pragma unroll
        for (int k = 0; k <= N; ++k) {
            const double w = row[colo[k]];
#pragma unroll
            for (int t = 0; t < NT; ++t) acc[t][k] = a[t] * w;
        }
#pragma unroll
        for (int tp = 0; tp < B; ++tp) {
            const double w = row[tp * WE];
#pragma unroll
            for (int t = 0; t < NT; ++t) accT[t][tp] = ((t >> tp) & 1) ? 0.0 : a[t] * w;
        }
    }
    // ---- phase 1b: sources in Q, streamed from the level buffer ----
    {
        int rec = x;
        for (int i = 0; i < L.j; ++i) {
            const int v = (int)(srcs & 15u);
            srcs >>= 4;
            const RecPtr<C> rp(sm + L.off_cur, rec);
            rec += L.cnt;
            const double* row = Wl + v * rowstride;
            double a[NT];
            team_load_rec<C>(rp, a);
#pragma unroll
            for (int k = 0; k <= N; ++k) {
                const double w = row[colo[k]];
#pragma unroll
                for (int t = 0; t < NT; ++t) acc[t][k] = fma(a[t], w, acc[t][k]);
            }
#pragma unroll
            for (int tp = 0; tp < B; ++tp) {
                const double w = row[tp * WE];
#pragma unroll
                for (int t = 0; t < NT; ++t)
                    if (!((t >> tp) & 1)) accT[t][tp] = fma(a[t], w, accT[t][tp]);
            }
        }
    }
    // ---- phase 2a: transitions inside T, by |R_T| (node (R_T + tp, tp) = accT[R_T][tp]) ----
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
                    if (!((t >> tp) & 1)) accT[t][tp] = fma(s, Wl[(ts * n + tp) * WE], accT[t][tp]);
            }
        }
    // ---- phase 2b: sources in T -> Q-targets and the close ----
#pragma unroll
    for (int k = 0; k <= N; ++k)
#pragma unroll
        for (int ts = 0; ts < B; ++ts) {
            const double w = Wl[ts * rowstride + colo[k]];
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if ((t >> ts) & 1) acc[t][k] = fma(accT[t ^ (1 << ts)][ts], w, acc[t][k]);
        }
    // ---- outputs: next-level records, and Z[(SQ, R_T)] = lf * close (lf = -1 per closed fermion loop) ----
#pragma unroll
    for (int k = 0; k < N; ++k) {
        if (orec[k] == 0xffff) continue;
        const RecPtr<C> o(sm + L.off_nxt, orec[k]);
#pragma unroll
        for (int p = 0; p < 4; ++p)
            *reinterpret_cast<double2*>(o.part(p)) = make_double2(acc[2 * p][k], acc[2 * p + 1][k]);
    }
    {
        const RecPtr<C> o(sm + L.off_z, L.lvlZ_j1 + x);
#pragma unroll
        for (int p = 0; p < 4; ++p)
            *reinterpret_cast<double2*>(o.part(p)) = make_double2(L.lf * acc[2 * p][N], L.lf * acc[2 * p + 1][N]);
    }
}

// Column item: ONE column k (Q-target k < Nown, or the close k == Nown) of pattern S_Q.  Used for the first levels,
// where a pattern has few sources but many targets: the whole-pattern item is then a long serial instruction
// stream on a handful of lanes while the other warps wait at the level barrier.  Every column thread repeats the
// T-target part (12 of its 20 FMAs per source), which costs FP64 issue slots nobody else wants at these levels
// and cuts the critical path of the level by the number of columns.
template <int C>
__device__ __forceinline__ void team_item_col(const TeamLevel& L, const uint32_t* dsc, int x, int k, double* sm,
                                              const double* Wl)
{
    using Lay = TeamLayout<C>;
    constexpr int WE = Lay::WE, NT = kTeamNT, B = kTeamB;
    const int n = L.n;
    const uint32_t w0 = dsc[0], w4 = dsc[4];
    unsigned srcs = dsc[5];
    const int zrec = (int)(w0 >> 16);
    const int h = (int)((w4 >> 24) & 15u);
    const int nown = (int)(w4 >> 28);
    const bool close = (k == nown);
    const int colo = (close ? h : (int)((w4 >> (4 * k)) & 15u)) * WE;
    const int rowstride = n * WE;
    double acc[NT], accT[NT][B];
    {
        const RecPtr<C> zp(sm + L.off_z, zrec);
        double a[NT];
        team_load_rec<C>(zp, a);
        const double* row = Wl + h * rowstride;
        const double w = row[colo];
#pragma unroll
        for (int t = 0; t < NT; ++t) acc[t] = a[t] * w;
#pragma unroll
        for (int tp = 0; tp < B; ++tp) {
            const double wt = row[tp * WE];
#pragma unroll
            for (int t = 0; t < NT; ++t) accT[t][tp] = ((t >> tp) & 1) ? 0.0 : a[t] * wt;
        }
    }
    {
        int rec = x;
        for (int i = 0; i < L.j; ++i) {
            const int v = (int)(srcs & 15u);
            srcs >>= 4;
            const RecPtr<C> rp(sm + L.off_cur, rec);
            rec += L.cnt;
            const double* row = Wl + v * rowstride;
            double a[NT];
            team_load_rec<C>(rp, a);
            const double w = row[colo];
#pragma unroll
            for (int t = 0; t < NT; ++t) acc[t] = fma(a[t], w, acc[t]);
#pragma unroll
            for (int tp = 0; tp < B; ++tp) {
                const double wt = row[tp * WE];
#pragma unroll
                for (int t = 0; t < NT; ++t)
                    if (!((t >> tp) & 1)) accT[t][tp] = fma(a[t], wt, accT[t][tp]);
            }
        }
    }
#pragma unroll
    for (int l = 1; l < B; ++l)
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            if (cpopc(t) != l) continue;
#pragma unroll
            for (int ts = 0; ts < B; ++ts) {
                if (!((t >> ts) & 1)) continue;
                const double sv = accT[t ^ (1 << ts)][ts];
#pragma unroll
                for (int tp = 0; tp < B; ++tp)
                    if (!((t >> tp) & 1)) accT[t][tp] = fma(sv, Wl[(ts * n + tp) * WE], accT[t][tp]);
            }
        }
#pragma unroll
    for (int ts = 0; ts < B; ++ts) {
        const double w = Wl[ts * rowstride + colo];
#pragma unroll
        for (int t = 0; t < NT; ++t)
            if ((t >> ts) & 1) acc[t] = fma(accT[t ^ (1 << ts)][ts], w, acc[t]);
    }
    const double sg = close ? L.lf : 1.0;             // Z = lf * close (lf = -1 per closed fermion loop)
    const int orec = close ? L.lvlZ_j1 + x : (int)reinterpret_cast<const uint16_t*>(dsc + 1)[k];
    const RecPtr<C> o(sm + (close ? L.off_z : L.off_nxt), orec);
#pragma unroll
    for (int p = 0; p < 4; ++p)
        *reinterpret_cast<double2*>(o.part(p)) = make_double2(sg * acc[2 * p], sg * acc[2 * p + 1]);
}

template <int C>
__device__ __forceinline__ void team_dispatch_item(const TeamLevel& L, const uint32_t* dsc, int x, double* sm,
                                                   const double* Wl, bool active)
{
    // warp-uniform target count: the widest item of the warp (all 32 lanes call this)
    const int Nown = active ? (int)(dsc[4] >> 28) : 0;
    const int N = __reduce_max_sync(0xffffffffu, Nown);
    if (!active) return;
    switch (N) {
        case 0: team_item<C, 0>(L, dsc, x, sm, Wl); break;
        case 1: team_item<C, 1>(L, dsc, x, sm, Wl); break;
        case 2: team_item<C, 2>(L, dsc, x, sm, Wl); break;
        case 3: team_item<C, 3>(L, dsc, x, sm, Wl); break;
        case 4: team_item<C, 4>(L, dsc, x, sm, Wl); break;
        case 5: team_item<C, 5>(L, dsc, x, sm, Wl); break;
        default: team_item<C, 6>(L, dsc, x, sm, Wl); break;
    }
}

// Z[(SQ = {}, R_T)] for the 8 subsets of T (stages h < 3), one thread per instance, in the propagation's own
// order (start / extend / close).  zr points at Z record 0 of this instance (already offset by g * 2).
template <int C>
__device__ __forceinline__ void team_small_stages(const double* Wl, int n, double* zr, double lf)
{
    using Lay = TeamLayout<C>;
    constexpr int WE = Lay::WE, PART = Lay::PART;
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
    for (int t = 0; t < 8; t += 2) *reinterpret_cast<double2*>(zr + (t >> 1) * PART) = make_double2(z[t], z[t + 1]);   // record 0: no swizzle
}

// ------------------------------------------------------------------------------------------ a4
// Connected reduction on configuration-interleaved blocks (reading R5; paper's Ref. [9]):
//   C'[S'] = D0[S'] - sum_{T' proper subset of S'} C'[T'] * D1[S' \ T'],   S' subset of vertices 1..n-1,
//   D0[S'] = D[S' + {0}] (array CB, becomes C' in place), D1[U] = D[U] (array DB).
// S' = (hi, lo), lo = the 4 lowest bits.  Row hi of an array holds the 16 lo-values of every configuration:
//   [part 0..7][configuration 0..NC-1][2 doubles], the part index XOR-ed with a fold of hi when a quarter warp
//   spans several rows (NC < 8).  A leaf multiplies block C'[T_hi] with block D1[S_hi \ T_hi] as a subset
//   convolution over lo (81 FMAs on 32 loaded values).  The 2^|S_hi| terms of one output are split over 2^s
//   lanes of one warp (lane bit k owns the k-th lowest vertex of S_hi), partial blocks are summed by a
//   recursive-halving shuffle exchange, and the diagonal block (T_hi = S_hi) is solved in registers.
// Block barrier of the team / pair kernels (every thread of the CTA is a compute thread).
__device__ __forceinline__ void team_sync(int) { __syncthreads(); }
#ifdef COS_PHASE_TIMING
#define COS_PHASE_MARK_T(k, nthr) do { team_sync(nthr); if (threadIdx.x == 0) { const long long now__ = clock64(); \
    atomicAdd(&g_phase_cycles[k], (unsigned long long)(now__ - phase_t0__)); phase_t0__ = now__; } } while (0)
#else
#define COS_PHASE_MARK_T(k, nthr) do { } while (0)
#endif

template <int NC> struct RedLayout {
    static constexpr int ROW = 16 * NC;
    static constexpr int PSTR = 2 * NC;
    static constexpr int MASK = (NC >= 8) ? 0 : (8 / NC - 1);
    static constexpr int SMAX = (NC >= 32) ? 0 : (NC == 16 ? 1 : (NC == 8 ? 2 : (NC == 4 ? 3 : (NC == 2 ? 4 : 5))));
};

template <int NC>
__device__ __forceinline__ int red_swz(unsigned hi)
{
    if (RedLayout<NC>::MASK == 0) return 0;
    return (int)((__popc(hi) & 1) | ((hi ^ (hi >> 2) ^ (hi >> 4)) & 2u)) & RedLayout<NC>::MASK;
}

// element lo of configuration cg in row hi (double offset relative to the array)
template <int NC>
__device__ __forceinline__ int red_elem(unsigned hi, unsigned lo, int cg)
{
    using R = RedLayout<NC>;
    return (int)hi * R::ROW + (int)((lo >> 1) ^ (unsigned)red_swz<NC>(hi)) * R::PSTR + cg * 2 + (int)(lo & 1u);
}

template <int NC>
__device__ __forceinline__ void red_load_block(const double* arr, unsigned hi, int cg, double (&v)[16])
{
    using R = RedLayout<NC>;
    const double* row = arr + (int)hi * R::ROW + cg * 2;
    const int sw = red_swz<NC>(hi);
#pragma unroll
    for (int p = 0; p < 8; ++p) {
        const double2 x = *reinterpret_cast<const double2*>(row + (p ^ sw) * R::PSTR);
        v[2 * p] = x.x;
        v[2 * p + 1] = x.y;
    }
}

template <int NC>
__device__ __forceinline__ void team_reduce(double* CB, double* DB, int ncfg, int n, const uint16_t* mask16,
                                            const int* lvlT, int tid, int nthreads)
{
    using R = RedLayout<NC>;
    const int hb = n - 1 - kRedLB;
    const int cg = tid % NC, slot = tid / NC, slots = nthreads / NC;
    // ---- make the diagonal block the identity: with g = (D1[hi = {}])^-1 (subset-convolution inverse over lo),
    //      C' = D0 / D1 = (D0 * g) / (D1 * g) and (D1 * g)[hi = {}] = delta, so that C'[S_hi] needs no triangular
    //      solve of its own -- the 65 dependent FMAs per output row leave the critical path of every level.
    //      Cost: one lo-convolution per row of both arrays, all rows in parallel. ----
    if (slot == 0 && cg < ncfg) {
        double e[16], gi[16];
        red_load_block<NC>(DB, 0u, cg, e);
        gi[0] = 1.0;                                      // D[{}] = 1
#pragma unroll
        for (int lo = 1; lo < 16; ++lo) {
            double v = 0.0;
#pragma unroll
            for (int T = 0; T < 16; ++T)
                if ((T & ~lo) == 0 && T != lo) v = fma(-gi[T], e[lo ^ T], v);
            gi[lo] = v;
        }
        double* row = DB + cg * 2;
#pragma unroll
        for (int p = 0; p < 8; ++p) *reinterpret_cast<double2*>(row + p * R::PSTR) = make_double2(gi[2 * p], gi[2 * p + 1]);   // row 0: no swizzle
    }
    team_sync(nthreads);
    {
        const int rows = 1 << hb;
        if (cg < ncfg) {
            double gi[16];
            red_load_block<NC>(DB, 0u, cg, gi);
            for (int task = slot; task < 2 * rows - 1; task += slots) {
                double* arr = task < rows ? CB : DB;
                const unsigned hi = (unsigned)(task < rows ? task : task - rows + 1);
                double v[16], o[16];
                red_load_block<NC>(arr, hi, cg, v);
#pragma unroll
                for (int t = 0; t < 16; ++t) o[t] = 0.0;
                leaf_conv(v, gi, o);
                double* row = arr + (int)hi * R::ROW + cg * 2;
                const int sw = red_swz<NC>(hi);
#pragma unroll
                for (int p = 0; p < 8; ++p)
                    *reinterpret_cast<double2*>(row + (p ^ sw) * R::PSTR) = make_double2(o[2 * p], o[2 * p + 1]);
            }
        }
    }
    team_sync(nthreads);
    for (int l = 1; l <= hb; ++l) {
        const int outputs = kBinom.c[hb][l];
        int s = l < R::SMAX ? l : R::SMAX;
        if (l == hb) {                     // top row: a plain butterfly sums one value, so a whole warp may share it
            constexpr int SFULL = NC >= 32 ? 0 : (NC == 16 ? 1 : (NC == 8 ? 2 : (NC == 4 ? 3 : (NC == 2 ? 4 : 5))));
            s = l < SFULL ? l : SFULL;
        }
        while (s > 0 && (outputs << s) > slots) --s;
        const int per_pass = slots >> s;
        const unsigned c = (unsigned)slot & ((1u << s) - 1u);
        for (int base = 0; base < outputs; base += per_pass) {
            const int o = base + (slot >> s);
            const bool active = (o < outputs) && (cg < ncfg) && ((slot >> s) < per_pass);
            double acc[16];
#pragma unroll
            for (int t = 0; t < 16; ++t) acc[t] = 0.0;
            unsigned S = 0;
            if (active) {
                S = mask16[lvlT[l] + o];
                unsigned tl = 0, m = S;
                for (int k = 0; k < s; ++k) {            // lane bit k owns the k-th lowest vertex of S
                    const unsigned bit = m & (0u - m);
                    m ^= bit;
                    if ((c >> k) & 1u) tl |= bit;
                }
                const unsigned rest = m;
                unsigned Th = rest;
                while (true) {
                    const unsigned T = Th | tl;
                    if (T != S) {
                        double cb[16], db[16];
                        red_load_block<NC>(CB, T, cg, cb);
                        red_load_block<NC>(DB, S ^ T, cg, db);
                        if (l == hb) {
                            // top row: only C'[full] = element lo = 15 is ever read (a5), 16 of the 81 products
                            double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
#pragma unroll
                            for (int t = 0; t < 16; t += 4) {
                                p0 = fma(cb[t], db[15 ^ t], p0);
                                p1 = fma(cb[t + 1], db[15 ^ (t + 1)], p1);
                                p2 = fma(cb[t + 2], db[15 ^ (t + 2)], p2);
                                p3 = fma(cb[t + 3], db[15 ^ (t + 3)], p3);
                            }
                            acc[15] += (p0 + p1) + (p2 + p3);
                        } else {
                            leaf_conv(cb, db, acc);
                        }
                    }
                    if (Th == 0) break;
                    Th = (Th - 1) & rest;
                }
            }
            if (l == hb) {
                // one value per lane: plain butterfly sum over the 2^s lanes of the output, then C'[full] -= sum
                double v = acc[15];
                for (int k = 0; k < s; ++k) v += __shfl_xor_sync(0xffffffffu, v, (NC << k) & 31);
                if (active && c == 0) { const int e = red_elem<NC>(S, 15u, cg); CB[e] = CB[e] - v; }
                continue;
            }
            // ---- sum the 2^s partial blocks: recursive halving, lane bit k keeps lo-bit k == its own bit ----
            double* blk = CB;     // element lo at blk[red_elem(S, lo, cg)]
            if (s == 0) {
                if (active) {
                    double* row = CB + (int)S * R::ROW + cg * 2;
                    const int sw = red_swz<NC>(S);
#pragma unroll
                    for (int p = 0; p < 8; ++p) {
                        double2* q2 = reinterpret_cast<double2*>(row + (p ^ sw) * R::PSTR);
                        const double2 d0 = *q2;
                        *q2 = make_double2(d0.x - acc[2 * p], d0.y - acc[2 * p + 1]);
                    }
                }
            } else {
                double r8[8];
                const bool b0 = c & 1u;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const double keep = sel(b0, acc[2 * i + 1], acc[2 * i]);
                    const double send = sel(b0, acc[2 * i], acc[2 * i + 1]);
                    r8[i] = keep + __shfl_xor_sync(0xffffffffu, send, NC);
                }
                if (s == 1) {
                    if (active) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) { const int e = red_elem<NC>(S, 2 * i + (int)b0, cg); blk[e] = blk[e] - r8[i]; }
                    }
                } else {
                    double r4[4];
                    const bool b1 = (c >> 1) & 1u;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const double keep = sel(b1, r8[2 * i + 1], r8[2 * i]);
                        const double send = sel(b1, r8[2 * i], r8[2 * i + 1]);
                        r4[i] = keep + __shfl_xor_sync(0xffffffffu, send, (NC * 2) & 31);
                    }
                    if (s == 2) {
                        if (active) {
#pragma unroll
                            for (int i = 0; i < 4; ++i) { const int e = red_elem<NC>(S, 4 * i + (int)(c & 3u), cg); blk[e] = blk[e] - r4[i]; }
                        }
                    } else {
                        double r2[2];
                        const bool b2 = (c >> 2) & 1u;
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const double keep = sel(b2, r4[2 * i + 1], r4[2 * i]);
                            const double send = sel(b2, r4[2 * i], r4[2 * i + 1]);
                            r2[i] = keep + __shfl_xor_sync(0xffffffffu, send, (NC * 4) & 31);
                        }
                        if (s == 3) {
                            if (active) {
#pragma unroll
                                for (int i = 0; i < 2; ++i) { const int e = red_elem<NC>(S, 8 * i + (int)(c & 7u), cg); blk[e] = blk[e] - r2[i]; }
                            }
                        } else {
                            const bool b3 = (c >> 3) & 1u;
                            const double keep = sel(b3, r2[1], r2[0]);
                            const double send = sel(b3, r2[0], r2[1]);
                            double r1 = keep + __shfl_xor_sync(0xffffffffu, send, (NC * 8) & 31);
                            if (s == 5) r1 += __shfl_xor_sync(0xffffffffu, r1, (NC * 16) & 31);   // NC == 1 only
                            if (active && !(c & 16u)) { const int e = red_elem<NC>(S, c & 15u, cg); blk[e] = blk[e] - r1; }
                        }
                    }
                }
            }
        }
        team_sync(nthreads);
    }
}

// a3: D[S] = w(S) Zup[S] Zdn[S] for the NC configurations of the team, written straight into the reduction
// arrays: S odd -> CB (D0[S >> 1]), S even -> DB (D1[S >> 1]).  One thread per (Z record, configuration): the 8
// values R_T of record S_Q are the lo-values (S_Q & 3) * 4 + {0..3} of row hi = S_Q >> 2 in both arrays.
// un[v * NC + cg] = -u_v of configuration cg (aliased species only; otherwise -u is folded into W).
template <int C, int NC>
__device__ __forceinline__ void team_combine(double* smd, const TeamDims& d, int ncfg, const uint16_t* recSQ,
                                             int tid, int nthreads)
{
    using Lay = TeamLayout<C>;
    using R = RedLayout<NC>;
    constexpr int NSP = C / NC;
    double* CB = smd + d.off_cb;
    double* DB = smd + d.off_db;
    const double* un = smd + d.off_u;
    const int cg = tid % NC;
    double wT[8];
#pragma unroll
    for (int t = 0; t < 8; ++t) wT[t] = 1.0;
    {
        const double u0 = un[0 * NC + cg], u1 = un[1 * NC + cg], u2 = un[2 * NC + cg];
#pragma unroll
        for (int t = 0; t < 8; ++t) wT[t] = ((t & 1) ? u0 : 1.0) * ((t & 2) ? u1 : 1.0) * ((t & 4) ? u2 : 1.0);
    }
    // w(S_Q) = wt[S_Q & 15] * wt[16 + (S_Q >> 4)]: products over the 4 low / 3 high vertices of Q, built once per team
    double* wt = smd + d.off_u + 16 * NC;
    {
        for (int t = tid / NC; t < 24; t += nthreads / NC) {
            unsigned m = t < 16 ? (unsigned)t : (unsigned)(t - 16) << 4;
            double w = 1.0;
            while (m) { const int v = __ffs(m) - 1; m &= m - 1; if (v < d.qmax) w *= un[(v + kTeamB) * NC + cg]; }
            wt[t * NC + cg] = w;
        }
        team_sync(nthreads);
    }
    for (int rec = tid / NC; rec < d.zrec; rec += nthreads / NC) {
        const unsigned SQ = recSQ[rec];
        const double wq = wt[(SQ & 15u) * NC + cg] * wt[(16u + (SQ >> 4)) * NC + cg];
        const RecPtr<C> zp(smd + d.off_z + (cg * NSP) * 2, rec);
        double val[8];
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const double2 zu = *reinterpret_cast<const double2*>(zp.part(p));
            const double2 zd = *reinterpret_cast<const double2*>(zp.part(p) + (NSP - 1) * 2);
            val[2 * p] = (wq * wT[2 * p]) * (zu.x * zd.x);
            val[2 * p + 1] = (wq * wT[2 * p + 1]) * (zu.y * zd.y);
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

// ---- inputs of one team: G (materialised by cos_build_G or by the caller) and the couplings ----
// The matrices of the NEXT team are fetched with cp.async into a staging buffer while the current team is being
// evaluated (stage[gi * n*n + e], coalesced rows of G; then u[cg * n + v] when per-vertex couplings are given), and
// unpacked into the replicated, instance-interleaved W at the start of the team:
//   W[e * (REP * C) + r * C + gi],  -u_a folded into the rows of species 0 when the species are distinct,
//   un[v * NCt + cg] = -u_v otherwise (w(S) is then applied in the combine step).
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <int C>
__device__ __forceinline__ void team_prefetch_inputs(const EvalArgs& a, int n, int nsp, double* stage, long long inst0,
                                                     int ninst, int tid, int nthreads)
{
    const int nn = n * n;
    for (int t = tid; t < ninst * nn; t += nthreads) {
        const int gi = t / nn, e = t - gi * nn;
        const long long b = (inst0 + gi) >> (nsp - 1);            // nsp is 1 or 2
        const int s = (int)((inst0 + gi) & (nsp - 1));
        cp_async8(stage + t, (s == 0 ? a.Gup : a.Gdn) + b * nn + e);
    }
    if (a.u) {
        const long long cfg0 = inst0 >> (nsp - 1);
        const int ncfg = ninst >> (nsp - 1);
        for (int t = tid; t < ncfg * n; t += nthreads) cp_async8(stage + C * nn + t, a.u + cfg0 * n + t);
    }
    cp_async_commit();
}

template <int C, int REP>
__device__ __forceinline__ void team_unpack_inputs(const EvalArgs& a, int n, int nsp, const double* stage, double* Wd,
                                                   double* un, int ninst, int tid, int nthreads)
{
    constexpr int WE = REP * C;
    const int nn = n * n;
    const int NCt = C / nsp, ncfg = ninst / nsp;
    const double* su = stage + C * nn;
    for (int t = tid; t < C * nn; t += nthreads) {
        const int gi = t % C, e = t / C;
        double val = 0.0;
        if (gi < ninst) {
            val = stage[gi * nn + e];
            if (nsp == 2 && (gi & 1) == 0) val *= -(a.u ? su[(gi >> 1) * n + e / n] : a.U);
        }
        double* w = Wd + e * WE + gi;
#pragma unroll
        for (int r = 0; r < REP; ++r) w[r * C] = val;
    }
    if (nsp == 1)
        for (int t = tid; t < NCt * n; t += nthreads) {
            const int cg = t % NCt, v = t / NCt;
            un[t] = (cg < ncfg) ? -(a.u ? su[cg * n + v] : a.U) : 0.0;
        }
}

// All per-order tables of the team kernel, into the table area at the start of shared memory (layout: TeamDims).
__device__ __forceinline__ void team_build_tables(unsigned char* smem_raw, const TeamDims& d, int tid, int nthreads)
{
    const int n = d.n, qmax = d.qmax;
    uint16_t* mask16 = reinterpret_cast<uint16_t*>(smem_raw);
    uint16_t* rank16 = mask16 + (1 << (d.n - 1));
    int* lvlT = reinterpret_cast<int*>(rank16 + (1 << (d.n - 1)));
    int* lvlZ = lvlT + 32;
    uint16_t* recSQ = reinterpret_cast<uint16_t*>(lvlZ + 32);
    // ---- tables: subsets of {0..n-2} by popcount in colex order (rank independent of the ground set) ----
    if (tid == 0) {
        int run = 0;
        for (int j = 0; j <= n; ++j) { lvlT[j] = run; run += kBinom.c[n - 1][j]; }
        run = 0;
        for (int j = 0; j <= qmax + 1; ++j) { lvlZ[j] = run; run += kBinom.c[qmax][j]; }
    }
    __syncthreads();
    for (unsigned mk = tid; mk < (1u << (n - 1)); mk += nthreads) {
        int rk = 0, i = 0;
        unsigned m = mk;
        while (m) { const int s = __ffs(m) - 1; m &= m - 1; ++i; rk += kBinom.c[s][i]; }
        rank16[mk] = (uint16_t)rk;
        mask16[lvlT[i] + rk] = (uint16_t)mk;
        if (mk < (1u << qmax)) recSQ[lvlZ[i] + rk] = (uint16_t)mk;
    }
    __syncthreads();
    uint32_t* dtab = reinterpret_cast<uint32_t*>(smem_raw + d.dsc_off);
    for (int r = 1 + tid; r < (1 << qmax); r += nthreads) team_build_descriptor(dtab + r * 8, recSQ[r], qmax, lvlZ, rank16);
    // column units (pattern x | column << 8) of level 0, their count in ucol[254]
    uint16_t* ucol = reinterpret_cast<uint16_t*>(smem_raw + d.dsc_off + 32 * d.zrec);
    __syncthreads();
    if (tid == 0) {
        int u = 0;
        for (int j = 0; j < 1; ++j) {
            for (int x = 0; x < kBinom.c[qmax][j + 1]; ++x) {
                const int nown = (int)(dtab[(lvlZ[j + 1] + x) * 8 + 4] >> 28);
                for (int k = 0; k <= nown && u < 254; ++k) ucol[u++] = (uint16_t)(x | (k << 8));
            }
            ucol[254 + j] = (uint16_t)u;
        }
    }

    __syncthreads();
}

// Builds the table image of one order once (one CTA); the evaluation kernels copy it instead of rebuilding it
// per CTA (the construction costs about 12 k cycles, a quarter of a whole order-8 launch at batch 4096).
__global__ void __launch_bounds__(256) team_tables_kernel(TeamDims d, unsigned char* out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    team_build_tables(smem_raw, d, threadIdx.x, blockDim.x);
    const uint4* src = reinterpret_cast<const uint4*>(smem_raw);
    uint4* dst = reinterpret_cast<uint4*>(out);
    for (int i = threadIdx.x; i < d.tab_bytes / 16; i += blockDim.x) dst[i] = src[i];
}

// Team kernel: the next team's matrices go straight into the replicated W with cp.async, issued as soon as the
// last propagation level has released W (the combine and the reduction do not read it), so that a team starts with
// its W in place -- no staging pass.  Only the couplings (a few values) are staged.
template <int C, int REP>
__device__ __forceinline__ void team_prefetch_w(const EvalArgs& a, int n, int nsp, double* Wd, double* stage_u,
                                                long long inst0, int ninst, int tid, int nthreads)
{
    // nthreads is a multiple of C: a thread always serves the same instance gi, and the entries e0, e0 + step, ..
    constexpr int WE = REP * C;
    const int nn = n * n;
    const int gi = tid % C, e0 = tid / C, step = nthreads / C;
    double* w = Wd + gi;
    if (gi < ninst) {
        const long long b = (inst0 + gi) >> (nsp - 1);                // nsp is 1 or 2
        const double* src = (((inst0 + gi) & (nsp - 1)) == 0 ? a.Gup : a.Gdn) + b * nn;
        for (int e = e0; e < nn; e += step) cp_async8(w + e * WE, src + e);      // replica 0; team_replicate_w copies it
    } else {
        for (int e = e0; e < nn; e += step) {
#pragma unroll
            for (int r = 0; r < REP; ++r) w[e * WE + r * C] = 0.0;
        }
    }
    if (a.u) {
        const long long cfg0 = inst0 >> (nsp - 1);
        const int ncfg = ninst >> (nsp - 1);
        for (int t = tid; t < ncfg * n; t += nthreads) cp_async8(stage_u + t, a.u + cfg0 * n + t);
    }
    cp_async_commit();
}

// Replicas 1..REP-1 of W from replica 0 (each thread copies the entries it fetched itself: no barrier in between).
template <int C, int REP>
__device__ __forceinline__ void team_replicate_w(int n, double* Wd, int ninst, int tid, int nthreads)
{
    constexpr int WE = REP * C;
    if (REP == 1) return;
    const int nn = n * n;
    const int gi = tid % C, e0 = tid / C, step = nthreads / C;
    if (gi >= ninst) return;
    double* w = Wd + gi;
    for (int e = e0; e < nn; e += step) {
        const double v = w[e * WE];
#pragma unroll
        for (int r = 1; r < REP; ++r) w[e * WE + r * C] = v;
    }
}

// un[v * NCt + cg] = -u_v of configuration cg of the team (0 for empty slots)
template <int C>
__device__ __forceinline__ void team_set_couplings(const EvalArgs& a, int n, int nsp, const double* stage_u, double* un,
                                                   int ninst, int tid, int nthreads)
{
    const int NCt = C / nsp, ncfg = ninst / nsp;
    for (int t = tid; t < NCt * n; t += nthreads) {
        const int cg = t % NCt, v = t / NCt;
        un[t] = (cg < ncfg) ? -(a.u ? stage_u[cg * n + v] : a.U) : 0.0;
    }
}

template <int C, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) eval_team_kernel(EvalArgs a, TeamDims d)
{
    using Lay = TeamLayout<C>;
    constexpr int WE = Lay::WE, REC = Lay::REC, PART = Lay::PART, REP = Lay::REP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
#ifdef COS_PHASE_TIMING
    long long phase_t0__ = clock64();
#endif
    uint16_t* mask16 = reinterpret_cast<uint16_t*>(smem_raw);
    uint16_t* rank16 = mask16 + (1 << (d.n - 1));
    int* lvlT = reinterpret_cast<int*>(rank16 + (1 << (d.n - 1)));   // list offsets, ground set n-1 bits
    int* lvlZ = lvlT + 32;                                           // Z record offsets, ground set qmax bits
    uint16_t* recSQ = reinterpret_cast<uint16_t*>(lvlZ + 32);        // Z record -> S_Q
    double* smd = reinterpret_cast<double*>(smem_raw + d.tab_bytes);
    const int tid = threadIdx.x, nthreads = blockDim.x;
    const int n = d.n, qmax = d.qmax, nsp = d.nsp;
    const unsigned NS = 1u << n;
    const long long total_inst = a.batch * nsp;
    const long long nteams = (total_inst + C - 1) / C;

    const int g = tid % C;                       // instance of this thread
    const int slot = tid / C;                    // pattern slot
    const int rep = slot % REP;                  // W replica read by this thread
    double* sm = smd + g * 2;
    const double* Wl = smd + d.off_w + rep * C + g;

    // the first team's inputs are fetched while the tables below are being built
    double* stage = smd + d.off_stage;
    if ((long long)blockIdx.x < nteams) {
        const long long nx0 = (long long)blockIdx.x * C;
        team_prefetch_w<C, REP>(a, n, nsp, smd + d.off_w, stage, nx0, (int)min((long long)C, total_inst - nx0), tid, nthreads);
    }
    // ---- tables (subset lists, ranks, item descriptors, column units): copied from the image the context built
    //      once per order (team_tables_kernel), or built here when no image is given ----
    uint32_t* dtab = reinterpret_cast<uint32_t*>(smem_raw + d.dsc_off);
    uint16_t* ucol = reinterpret_cast<uint16_t*>(smem_raw + d.dsc_off + 32 * d.zrec);
    if (a.tabs != nullptr) {
        const uint4* src = reinterpret_cast<const uint4*>(a.tabs);
        uint4* dst = reinterpret_cast<uint4*>(smem_raw);
        for (int i = tid; i < d.tab_bytes / 16; i += nthreads) dst[i] = __ldg(src + i);
    } else {
        team_build_tables(smem_raw, d, tid, nthreads);
    }

    const bool col_ok = qmax >= 2 && qmax <= 7;      // unit table: 28 + 91 entries at most (order 10)
    for (long long team = blockIdx.x; team < nteams; team += gridDim.x) {
        const long long inst0 = team * C;
        const int ninst = (int)min((long long)C, total_inst - inst0);
        const int ncfg = ninst / nsp;
        const int NCt = C / nsp;                 // configuration slots of a team
        const long long cfgbase = inst0 / nsp;
        cp_async_wait_all();
        team_replicate_w<C, REP>(n, smd + d.off_w, ninst, tid, nthreads);
        __syncthreads();          // W of this team is in place; the previous team's last reads are done
        team_set_couplings<C>(a, n, nsp, stage, smd + d.off_u, ninst, tid, nthreads);
        COS_PHASE_MARK_T(0, nthreads);
        if (tid < ninst) team_small_stages<C>(smd + d.off_w + tid, n, smd + d.off_z + tid * 2, a.loopf);
        team_sync(nthreads);
        COS_PHASE_MARK_T(1, nthreads);

        // ---- a2: all stages together, level j = |S_Q| - 1 ----
        TeamLevel L;
        L.n = n; L.rank16 = rank16; L.off_z = d.off_z; L.lf = a.loopf;
        int cur = d.off_b0, nxt = d.off_b1;
        for (int j = 0; j < qmax; ++j) {
            L.j = j;
            L.cnt = kBinom.c[qmax][j + 1];
            L.cnt_next = kBinom.c[qmax][j + 2];
            L.lvlZ_j = lvlZ[j]; L.lvlZ_j1 = lvlZ[j + 1];
            L.off_cur = cur; L.off_nxt = nxt;
            if (j == 0 && col_ok) {      // measured: column items win at level 0 only (level 1 needs three passes)
                const int ub = 0, ue = (int)ucol[254];
                for (int u0 = ub; u0 < ue; u0 += d.pslots) {
                    const int u = u0 + slot;
                    if (u < ue && g < ninst) {
                        const int xk = (int)ucol[u];
                        team_item_col<C>(L, dtab + (L.lvlZ_j1 + (xk & 255)) * 8, xk & 255, xk >> 8, sm, Wl);
                    }
                }
            } else
            for (int x0 = 0; x0 < L.cnt; x0 += d.pslots) {
                const int x = x0 + slot;
                const bool active = (x < L.cnt) && (g < ninst);
                team_dispatch_item<C>(L, dtab + (L.lvlZ_j1 + (active ? x : 0)) * 8, x, sm, Wl, active);
            }
            team_sync(nthreads);
            COS_PHASE_MARK_T(2 + j, nthreads);
            const int tmp = cur; cur = nxt; nxt = tmp;
        }

        // W is dead from here on: fetch the next team's matrices into it (the barrier of the last level is behind us;
        // the couplings of THIS team were copied out of the staging area before the levels)
        if (team + gridDim.x < nteams) {
            const long long nx0 = (team + gridDim.x) * C;
            team_prefetch_w<C, REP>(a, n, nsp, smd + d.off_w, stage, nx0, (int)min((long long)C, total_inst - nx0), tid, nthreads);
        }
        // ---- a3 + a5 ("all"): D[full] = w * Zup[full] * Zdn[full] ----
        if (!a.connected) {
            if (tid < ncfg) {
                const int rec = lvlZ[qmax];                            // S_Q = Q, R_T = T: part 3, second value
                const int part = Lay::SWZ ? (3 ^ (rec & 1)) : 3;
                const double* zp = smd + d.off_z + rec * REC + part * PART + 1;
                const double zu = zp[(tid * nsp) * 2];
                const double zd = zp[(tid * nsp + nsp - 1) * 2];
                double w = 1.0;
                for (int v = 0; v < n; ++v) w *= smd[d.off_u + v * NCt + tid];
                a.out[cfgbase + tid] = w * zu * zd;
            }
            continue;
        }

        // ---- a3: combine, a4: connected reduction, a5: C'[full] ----
        double* CB = smd + d.off_cb;
        double* DB = smd + d.off_db;
        if (nsp == 1) {
            team_combine<C, C>(smd, d, ncfg, recSQ, tid, nthreads);
            team_sync(nthreads);
            COS_PHASE_MARK_T(12, nthreads);
            team_reduce<C>(CB, DB, ncfg, n, mask16, lvlT, tid, nthreads);
            COS_PHASE_MARK_T(13, nthreads);
            if (tid < ncfg) a.out[cfgbase + tid] = CB[red_elem<C>((NS >> (1 + kRedLB)) - 1, 15u, tid)];
        } else {
            team_combine<C, C / 2>(smd, d, ncfg, recSQ, tid, nthreads);
            team_sync(nthreads);
            COS_PHASE_MARK_T(12, nthreads);
            team_reduce<C / 2>(CB, DB, ncfg, n, mask16, lvlT, tid, nthreads);
            COS_PHASE_MARK_T(13, nthreads);
            if (tid < ncfg) a.out[cfgbase + tid] = CB[red_elem<C / 2>((NS >> (1 + kRedLB)) - 1, 15u, tid)];
        }
    }
}

}  // namespace cosb
