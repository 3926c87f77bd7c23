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
//    half warp read different bank groups, so it is conflict free by construction as well.
//  * vertices are split into T = {0,1,2} and Q = {3..n-1} as in the tiled kernel: one thread carries the 8
//    subsets R_T of one Q-pattern, every W entry it loads is used 8 times, transitions inside T stay in
//    registers, and every FMA executed is one the method needs.
//  * ALL stages h advance together: level j holds every node (S, c) whose Q-part S_Q has j + 1 elements
//    (its top element is the stage vertex h).  Patterns of one level are the (j+1)-subsets of Q in colex
//    order -- which sorts by h first -- so there are only n - 3 block barriers per propagation instead of
//    (n-3)(n-2)/2, and a level exposes C(n-3, j+1) x C items of parallel work.
//  * the two species of one configuration are two instances of the same team, so G_up != G_dn costs no
//    extra shared memory per instance.
#pragma once
#include "cos_common.cuh"
#include "cos_kernels_generic.cuh"
#include "cos_kernels_tiled.cuh"   // kBinom, cpopc, reduce_blocked_rt

namespace cosb {

constexpr int kTeamB = 3;          // |T|
constexpr int kTeamNT = 8;         // 2^|T|
constexpr int kTeamMaxTargets = 6; // Q-targets held in registers per pass (orders <= 10 need at most 6)

template <int C> struct TeamLayout {
    static_assert(C == 8 || C == 16 || C == 32, "instances per team");
    static constexpr int REP = (C >= 16) ? 1 : 16 / C;   // W replicas
    static constexpr int WE = REP * C;                   // doubles per W entry
    static constexpr int PART = 2 * C;                   // doubles per record part
    static constexpr int REC = 8 * C;                    // doubles per node record
};

struct TeamDims {
    int n, nsp, C;
    int qmax;          // n - 3
    int pslots;        // pattern slots per pass = threads / C
    int threads;
    int maxrec;        // records per frontier buffer
    int zrec;          // Z records (2^qmax)
    int ncfg;          // configurations per team = C / nsp
    int red_stride;    // doubles per configuration of the reduction arrays
    int off_w, off_u, off_z, off_b0, off_b1;   // double offsets behind the tables
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
    const int lanes_pat = 32 / (C < 32 ? C : 32);         // patterns per warp
    int slots = team_max_patterns(n);
    slots = (slots + lanes_pat - 1) / lanes_pat * lanes_pat;
    d.pslots = slots;
    d.threads = slots * C;
    if (d.threads < 64) { d.threads = 64; d.pslots = 64 / C; }
    int maxrec = 1;
    for (int j = 0; j <= d.qmax; ++j) {
        const int v = j * kBinomHost.c[d.qmax][j + 1];
        if (v > maxrec) maxrec = v;
    }
    d.maxrec = maxrec;
    d.zrec = 1 << d.qmax;
    d.ncfg = C / nsp;
    d.red_stride = red_doubles(n) + 2;
    d.off_w = 0;
    d.off_u = d.off_w + n * n * L::WE;
    d.off_z = d.off_u + C * 64;                           // per configuration: wlo[32], whi[32]
    d.off_b0 = d.off_z + d.zrec * L::REC;
    int work = 2 * maxrec * L::REC;
    const int need = d.ncfg * d.red_stride;
    if (work < need) work = need;
    d.off_b1 = d.off_b0 + maxrec * L::REC;
    d.tab_bytes = ((2 * 2 * (1 << (n - 1)) + 4 * 64) + 15) & ~15;
    d.smem_bytes = (size_t)d.tab_bytes + sizeof(double) * (size_t)(d.off_b0 + work);
    return d;
}

// Uniform description of one level step.
struct TeamLevel {
    int n, j;
    int cnt, cnt_next;          // patterns at levels j and j + 1
    int lvlZ_j, lvlZ_j1;        // Z record offsets of |S_Q| = j and j + 1
    int off_z, off_cur, off_nxt;
    const uint16_t* rank16;
};

// One item: Q-pattern SQ (|SQ| = j + 1, top element q, stage vertex h = q + 3) of one instance.
//   sm : shared doubles, already offset by the instance (g * 2)
//   Wl : W of this instance and replica, entry (c, c') at Wl[(c * n + c') * WE]
// N = q - j Q-targets are accumulated in registers together with the close (column h) and the T-targets.
template <int C, int N>
__device__ __forceinline__ void team_item(const TeamLevel& L, unsigned SQ, int x, double* sm, const double* Wl)
{
    using Lay = TeamLayout<C>;
    constexpr int WE = Lay::WE, REC = Lay::REC, PART = Lay::PART, NT = kTeamNT, B = kTeamB;
    const int n = L.n;
    const int q = 31 - __clz((int)SQ);
    const unsigned RQ = SQ ^ (1u << q);
    const int h = q + B;
    int colo[N + 1];                  // W column offset of target k; the last one is the close column h
    int orec[N > 0 ? N : 1];          // double offset of target k's record in the next buffer
    {
        unsigned absent = ~RQ & ((1u << q) - 1u);
#pragma unroll
        for (int k = 0; k < N; ++k) {
            const int d = __ffs(absent) - 1;
            absent &= absent - 1;
            colo[k] = (d + B) * WE;
            orec[k] = (__popc(RQ & ((1u << d) - 1u)) * L.cnt_next + L.rank16[SQ | (1u << d)]) * REC;
        }
        colo[N] = h * WE;
    }
    double acc[NT][N + 1], accT[NT][B];
#pragma unroll
    for (int t = 0; t < NT; ++t) {
#pragma unroll
        for (int k = 0; k <= N; ++k) acc[t][k] = 0.0;
#pragma unroll
        for (int tp = 0; tp < B; ++tp) accT[t][tp] = 0.0;
    }
    // ---- phase 1: sources in Q (streamed from the level buffer) and the start node h (from Z) ----
    {
        const double* rec = sm + L.off_cur + x * REC;
        const int step = L.cnt * REC;
        const double* zsrc = sm + L.off_z + (L.lvlZ_j + L.rank16[RQ]) * REC;
        unsigned m = RQ;
        const int rowstride = n * WE;
        for (int i = 0; i <= L.j; ++i) {
            const double* p;
            int v;
            if (i < L.j) {
                v = __ffs(m) - 1 + B;
                m &= m - 1;
                p = rec;
                rec += step;
            } else {
                v = h;
                p = zsrc;
            }
            const double* row = Wl + v * rowstride;
            double a[NT];
#pragma unroll
            for (int t = 0; t < NT; t += 2) {
                const double2 v2 = *reinterpret_cast<const double2*>(p + (t >> 1) * PART);
                a[t] = v2.x;
                a[t + 1] = v2.y;
            }
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
            const double w = Wl[ts * n * WE + colo[k]];
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if ((t >> ts) & 1) acc[t][k] = fma(accT[t ^ (1 << ts)][ts], w, acc[t][k]);
        }
    // ---- outputs: next-level records, and Z[(SQ, R_T)] = -close (one -1 per closed fermion loop) ----
#pragma unroll
    for (int k = 0; k < N; ++k) {
        double* o = sm + L.off_nxt + orec[k];
#pragma unroll
        for (int t = 0; t < NT; t += 2)
            *reinterpret_cast<double2*>(o + (t >> 1) * PART) = make_double2(acc[t][k], acc[t + 1][k]);
    }
    {
        double* o = sm + L.off_z + (L.lvlZ_j1 + x) * REC;
#pragma unroll
        for (int t = 0; t < NT; t += 2)
            *reinterpret_cast<double2*>(o + (t >> 1) * PART) = make_double2(-acc[t][N], -acc[t + 1][N]);
    }
}

// Z[(SQ = {}, R_T)] for the 8 subsets of T (stages h < 3), one thread per instance, in the propagation's own
// order (start / extend / close).  zr points at Z record 0 of this instance (already offset by g * 2).
template <int C>
__device__ __forceinline__ void team_small_stages(const double* Wl, int n, double* zr)
{
    using Lay = TeamLayout<C>;
    constexpr int WE = Lay::WE, PART = Lay::PART;
    auto W = [&](int a, int b) { return Wl[(a * n + b) * WE]; };
    const double w00 = W(0, 0), w01 = W(0, 1), w02 = W(0, 2);
    const double w10 = W(1, 0), w11 = W(1, 1), w12 = W(1, 2);
    const double w20 = W(2, 0), w21 = W(2, 1), w22 = W(2, 2);
    double z[8];
    z[0] = 1.0;                                           // top node
    z[1] = -w00;                                          // stage 0
    z[2] = -w11;                                          // stage 1, R = {}
    z[3] = -fma(w10, w01, z[1] * w11);                    // stage 1, R = {0}: nodes (R,0) = W[1][0], (R,1) = Z[{0}]
    z[4] = -w22;                                          // stage 2, R = {}
    z[5] = -fma(w20, w02, z[1] * w22);                    // R = {0}
    z[6] = -fma(w21, w12, z[2] * w22);                    // R = {1}
    const double p01_1 = fma(w20, w01, z[1] * w21);       // node ({0,1}, 1) from R = {0}
    const double p01_0 = fma(w21, w10, z[2] * w20);       // node ({0,1}, 0) from R = {1}
    z[7] = -fma(p01_0, w02, fma(p01_1, w12, z[3] * w22)); // R = {0,1}
#pragma unroll
    for (int t = 0; t < 8; t += 2) *reinterpret_cast<double2*>(zr + (t >> 1) * PART) = make_double2(z[t], z[t + 1]);
}

template <int C>
__device__ __forceinline__ void team_dispatch_item(const TeamLevel& L, unsigned SQ, int x, double* sm, const double* Wl)
{
    const int N = (31 - __clz((int)SQ)) - L.j;
    switch (N) {
        case 0: team_item<C, 0>(L, SQ, x, sm, Wl); break;
        case 1: team_item<C, 1>(L, SQ, x, sm, Wl); break;
        case 2: team_item<C, 2>(L, SQ, x, sm, Wl); break;
        case 3: team_item<C, 3>(L, SQ, x, sm, Wl); break;
        case 4: team_item<C, 4>(L, SQ, x, sm, Wl); break;
        case 5: team_item<C, 5>(L, SQ, x, sm, Wl); break;
        default: team_item<C, 6>(L, SQ, x, sm, Wl); break;
    }
}

template <int C, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) eval_team_kernel(EvalArgs a, TeamDims d)
{
    using Lay = TeamLayout<C>;
    constexpr int WE = Lay::WE, REC = Lay::REC, PART = Lay::PART, REP = Lay::REP, B = kTeamB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint16_t* mask16 = reinterpret_cast<uint16_t*>(smem_raw);
    uint16_t* rank16 = mask16 + (1 << (d.n - 1));
    int* lvlT = reinterpret_cast<int*>(rank16 + (1 << (d.n - 1)));   // list offsets, ground set n-1 bits
    int* lvlZ = lvlT + 32;                                           // Z record offsets, ground set qmax bits
    double* smd = reinterpret_cast<double*>(smem_raw + d.tab_bytes);
    const int tid = threadIdx.x, nthreads = blockDim.x;
    const int n = d.n, qmax = d.qmax, nsp = d.nsp;
    const unsigned NS = 1u << n;
    const int g = tid % C;                       // instance of this thread
    const int slot = tid / C;                    // pattern slot
    const int rep = slot % REP;                  // W replica read by this thread
    double* sm = smd + g * 2;
    const double* Wl = smd + d.off_w + rep * C + g;

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
    }
    __syncthreads();

    const long long total_inst = a.batch * nsp;
    const long long nteams = (total_inst + C - 1) / C;
    for (long long team = blockIdx.x; team < nteams; team += gridDim.x) {
        const long long inst0 = team * C;
        const int ninst = (int)min((long long)C, total_inst - inst0);
        const int ncfg = ninst / nsp;
        const long long cfgbase = inst0 / nsp;
        __syncthreads();
        // ---- a1 (fused) / load: W of every instance, instance fastest; -u_a folded into the rows of species 0
        //      when the species are distinct.  Replica r of entry e lives at e*WE + r*C + g. ----
        for (int t = tid; t < C * n * n; t += nthreads) {
            const int gi = t % C, e = t / C;
            double val = 0.0;
            if (gi < ninst) {
                const long long b = (inst0 + gi) / nsp;
                const int s = (int)((inst0 + gi) % nsp);
                if (a.fused) {
                    double gu, gd;
                    g0_entry(a.bg, b, e / n, e % n, gu, gd);
                    val = s ? gd : gu;
                } else {
                    val = (s == 0 ? a.Gup : a.Gdn)[b * n * n + e];
                }
                if (nsp == 2 && s == 0) val *= -(a.u ? a.u[b * n + e / n] : a.U);
            }
            double* w = smd + d.off_w + e * WE + gi;
#pragma unroll
            for (int r = 0; r < REP; ++r) w[((r + e) % REP) * C] = val;
        }
        // w(S) = prod_{v in S} (-u_v) as wlo[S & 31] * whi[S >> 5] (aliased species only)
        if (nsp == 1) {
            for (int t = tid; t < ncfg * 64; t += nthreads) {
                const int cg = t >> 6, idx = t & 63, hi = idx >> 5;
                unsigned bits = (unsigned)(idx & 31);
                double w = 1.0;
                while (bits) {
                    const int v = __ffs(bits) - 1 + 5 * hi;
                    bits &= bits - 1;
                    if (v < n) w *= -(a.u ? a.u[(cfgbase + cg) * n + v] : a.U);
                }
                smd[d.off_u + cg * 64 + idx] = w;
            }
        }
        __syncthreads();
        if (tid < ninst) team_small_stages<C>(smd + d.off_w + tid, n, smd + d.off_z + tid * 2);
        __syncthreads();

        // ---- a2: all stages together, level j = |S_Q| - 1 ----
        TeamLevel L;
        L.n = n; L.rank16 = rank16; L.off_z = d.off_z;
        int cur = d.off_b0, nxt = d.off_b1;
        for (int j = 0; j < qmax; ++j) {
            L.j = j;
            L.cnt = kBinom.c[qmax][j + 1];
            L.cnt_next = kBinom.c[qmax][j + 2];
            L.lvlZ_j = lvlZ[j]; L.lvlZ_j1 = lvlZ[j + 1];
            L.off_cur = cur; L.off_nxt = nxt;
            const uint16_t* masks = mask16 + lvlT[j + 1];
            for (int x = slot; x < L.cnt; x += d.pslots)
                if (g < ninst) team_dispatch_item<C>(L, masks[x], x, sm, Wl);
            __syncthreads();
            const int tmp = cur; cur = nxt; nxt = tmp;
        }

        // ---- a3 + a5 ("all"): D[full] = w * Zup[full] * Zdn[full] ----
        if (!a.connected) {
            if (tid < ncfg) {
                const int full = lvlZ[qmax] * REC + 3 * PART + 1;      // S_Q = Q, R_T = T
                const double zu = smd[d.off_z + full + (tid * nsp) * 2];
                const double zd = smd[d.off_z + full + (tid * nsp + nsp - 1) * 2];
                double w = 1.0;
                if (nsp == 1) w = smd[d.off_u + tid * 64 + ((NS - 1) & 31)] * smd[d.off_u + tid * 64 + 32 + ((NS - 1) >> 5)];
                a.out[cfgbase + tid] = w * zu * zd;
            }
            continue;
        }

        // ---- a3: D[S] = w(S) Zup[S] Zdn[S], split by vertex 0 into D0[S'] = D[2S'+1] (becomes C' in place)
        //      and D1[U] = D[2U], both in the padded block layout of cos_reduce_blocked.cuh ----
        double* red = smd + d.off_b0;
        const int off_c = 0, off_d1 = red_rows(n) * kRowStride;
        for (unsigned t = tid; t < (unsigned)ncfg * NS; t += nthreads) {
            const unsigned cg = t % (unsigned)ncfg, S = t / (unsigned)ncfg;
            const unsigned SQ = S >> B, ST = S & 7u;
            const int at = d.off_z + (lvlZ[__popc(SQ)] + rank16[SQ]) * REC + (int)(ST >> 1) * PART + (int)(ST & 1u);
            const double zu = smd[at + (cg * nsp) * 2];
            const double zd = smd[at + (cg * nsp + nsp - 1) * 2];
            double w = 1.0;
            if (nsp == 1) w = smd[d.off_u + cg * 64 + (S & 31u)] * smd[d.off_u + cg * 64 + 32 + (S >> 5)];
            red[cg * d.red_stride + ((S & 1u) ? off_c : off_d1) + red_addr(S >> 1)] = w * zu * zd;
        }
        __syncthreads();

        // ---- a4: connected reduction, a5: C'[full] ----
        reduce_blocked_rt(red, d.red_stride, off_c, off_d1, ncfg, n, mask16, lvlT, tid, nthreads);
        if (tid < ncfg) a.out[cfgbase + tid] = red[tid * d.red_stride + off_c + red_addr((NS >> 1) - 1)];
    }
}

}  // namespace cosb
