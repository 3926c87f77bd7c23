// cos_reduce_blocked.cuh -- step a4, the connected reduction, register blocked.
//
//   C'[S'] = D0[S'] - sum_{T' proper subset of S'} C'[T'] * D1[S' \ T'],   S' subset of vertices 1..n-1,
//   D0[S'] = D[S' + {0}], D1[U] = D[U]  (paper's Ref. [9]; reading R5).
//
// S' = (hi, lo) with lo = the 4 lowest bits.  A "leaf" multiplies the 16-value block C'[T_hi, .] with the
// block D1[U_hi, .] as a subset convolution over lo: 81 FMAs on 32 loaded values, all in registers.
//   out[S_hi, .] = sum over T_hi subset of S_hi (T_hi != S_hi) of leaf(C'[T_hi], D1[S_hi \ T_hi])
// level by level in |S_hi|; the diagonal block (T_hi = S_hi) is made the identity beforehand (see the code).
// The 2^|S_hi| terms of one output are split over 2^s adjacent lanes (s chosen per level so that the CTA
// is filled); the lane owns the sub-subsets of s chosen vertices of S_hi, partial blocks are summed by a
// recursive-halving shuffle exchange.  Blocks are rows of 18 doubles (144 B) whose row index is XOR-folded
// so that the 8 lanes of one LDS.128 wavefront, which differ in three chosen vertices, hit 8 different
// 16-byte bank groups.
#pragma once
#include "cos_common.cuh"

namespace cosb {

constexpr int kLB = 4;            // lo bits held in registers
constexpr int kRowStride = 18;    // doubles per block row (16 + 2 padding)

__host__ __device__ __forceinline__ int red_phys_row(unsigned hi)
{
    return (int)((hi & ~7u) | ((hi ^ (hi >> 3) ^ (hi >> 6) ^ (hi >> 9)) & 7u));
}
__host__ __device__ inline int red_rows(int n) { return 1 << (n - 1 - kLB); }
__host__ __device__ inline int red_doubles(int n) { return 2 * red_rows(n) * kRowStride; }
// address (in doubles, relative to the array) of element S' = (hi << 4) | lo
__host__ __device__ __forceinline__ int red_addr(unsigned Sp) { return red_phys_row(Sp >> kLB) * kRowStride + (int)(Sp & 15u); }

__device__ __forceinline__ void load_block(const double* p, double (&v)[16])
{
#pragma unroll
    for (int t = 0; t < 16; t += 2) {
        const double2 x = *reinterpret_cast<const double2*>(p + t);
        v[t] = x.x;
        v[t + 1] = x.y;
    }
}

__device__ __forceinline__ void leaf_conv(const double (&c)[16], const double (&dd)[16], double (&acc)[16])
{
#pragma unroll
    for (int S = 0; S < 16; ++S)
#pragma unroll
        for (int T = 0; T < 16; ++T)
            if ((T & ~S) == 0) acc[S] = fma(c[T], dd[S ^ T], acc[S]);
}

__device__ __forceinline__ double sel(bool p, double a, double b) { return p ? a : b; }

// THREADS: threads of the CTA (a multiple of 32; all of them must call).
__device__ __forceinline__ void reduce_blocked_rt(double* cfg0, int cfg_doubles, int off_c, int off_d1, int ng, int n,
                                                  const uint16_t* mask16, const int* lvlT, int tid, const int THREADS)
{
    const int hb = n - 1 - kLB;
    // ---- identity diagonal block: with g = (D1[hi = {}])^-1 over lo, C' = (D0 * g) / (D1 * g) and
    //      (D1 * g)[hi = {}] = delta, so no output row needs a triangular solve of its own ----
    if (tid < ng) {
        double* Dg = cfg0 + (size_t)tid * cfg_doubles + off_d1;
        double e[16], gi[16];
        load_block(Dg, e);                               // red_phys_row(0) == 0
        gi[0] = 1.0;                                     // D[{}] = 1
#pragma unroll
        for (int lo = 1; lo < 16; ++lo) {
            double v = 0.0;
#pragma unroll
            for (int T = 0; T < 16; ++T)
                if ((T & ~lo) == 0 && T != lo) v = fma(-gi[T], e[lo ^ T], v);
            gi[lo] = v;
        }
#pragma unroll
        for (int t = 0; t < 16; t += 2) *reinterpret_cast<double2*>(Dg + t) = make_double2(gi[t], gi[t + 1]);
    }
    __syncthreads();
    {
        const int rows = 1 << hb;
        const int per_cfg = 2 * rows - 1;
        for (int task = tid; task < ng * per_cfg; task += THREADS) {
            const int g = task / per_cfg, r = task - g * per_cfg;
            double* base = cfg0 + (size_t)g * cfg_doubles;
            double* row = (r < rows) ? base + off_c + red_phys_row((unsigned)r) * kRowStride
                                     : base + off_d1 + red_phys_row((unsigned)(r - rows + 1)) * kRowStride;
            double gi[16], v[16], o[16];
            load_block(base + off_d1, gi);
            load_block(row, v);
#pragma unroll
            for (int t = 0; t < 16; ++t) o[t] = 0.0;
            leaf_conv(v, gi, o);
#pragma unroll
            for (int t = 0; t < 16; t += 2) *reinterpret_cast<double2*>(row + t) = make_double2(o[t], o[t + 1]);
        }
    }
    __syncthreads();
    for (int l = 1; l <= hb; ++l) {
        const int cntl = kBinom.c[hb][l];
        const int outputs = ng * cntl;
        int s = l < 5 ? l : 5;
        while (s > 0 && (outputs << s) > THREADS) --s;
        const int per_pass = THREADS >> s;
        const unsigned c = (unsigned)tid & ((1u << s) - 1u);
        for (int base = 0; base < outputs; base += per_pass) {
            const int o = base + (tid >> s);
            const bool active = o < outputs;
            double acc[16];
#pragma unroll
            for (int t = 0; t < 16; ++t) acc[t] = 0.0;
            double* Cg = cfg0;
            const double* Dg = cfg0;
            unsigned S = 0;
            if (active) {
                const int g = o / cntl, rr = o - g * cntl;
                S = mask16[lvlT[l] + rr];
                Cg = cfg0 + (size_t)g * cfg_doubles + off_c;
                Dg = cfg0 + (size_t)g * cfg_doubles + off_d1;
                // split vertices: first one per residue class mod 3 (distinct bank groups under the row fold),
                // then the lowest remaining ones; lane bit k owns the k-th chosen vertex
                unsigned chosen = 0, tl = 0, res = 0, m = S;
                int k = 0;
                while (m && k < s && k < 3) {
                    const unsigned bit = m & (0u - m);
                    m ^= bit;
                    const unsigned r = (unsigned)(__ffs(bit) - 1) % 3u;
                    if (!((res >> r) & 1u)) {
                        res |= 1u << r;
                        chosen |= bit;
                        if ((c >> k) & 1u) tl |= bit;
                        ++k;
                    }
                }
                m = S & ~chosen;
                while (k < s) {
                    const unsigned bit = m & (0u - m);
                    m ^= bit;
                    chosen |= bit;
                    if ((c >> k) & 1u) tl |= bit;
                    ++k;
                }
                const unsigned rest = S ^ chosen;
                unsigned Th = rest;
                while (true) {
                    const unsigned T = Th | tl;
                    if (T != S) {
                        double cb[16], db[16];
                        load_block(Cg + red_phys_row(T) * kRowStride, cb);
                        load_block(Dg + red_phys_row(S ^ T) * kRowStride, db);
                        leaf_conv(cb, db, acc);
                    }
                    if (Th == 0) break;
                    Th = (Th - 1) & rest;
                }
            }
            // ---- sum the 2^s partial blocks: recursive halving, lane bit k keeps lo-bit k == its own bit ----
            double* blk = Cg + red_phys_row(S) * kRowStride;
            if (s == 0) {
                if (active) {
#pragma unroll
                    for (int t = 0; t < 16; t += 2) {
                        const double2 d0 = *reinterpret_cast<const double2*>(blk + t);
                        *reinterpret_cast<double2*>(blk + t) = make_double2(d0.x - acc[t], d0.y - acc[t + 1]);
                    }
                }
            } else {
                double r8[8];
                const bool b0 = c & 1u;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const double keep = sel(b0, acc[2 * i + 1], acc[2 * i]);
                    const double send = sel(b0, acc[2 * i], acc[2 * i + 1]);
                    r8[i] = keep + __shfl_xor_sync(0xffffffffu, send, 1);
                }
                if (s == 1) {
                    if (active) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) { const int lo = 2 * i + (int)b0; blk[lo] = blk[lo] - r8[i]; }
                    }
                } else {
                    double r4[4];
                    const bool b1 = (c >> 1) & 1u;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const double keep = sel(b1, r8[2 * i + 1], r8[2 * i]);
                        const double send = sel(b1, r8[2 * i], r8[2 * i + 1]);
                        r4[i] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
                    }
                    if (s == 2) {
                        if (active) {
#pragma unroll
                            for (int i = 0; i < 4; ++i) { const int lo = 4 * i + (int)(c & 3u); blk[lo] = blk[lo] - r4[i]; }
                        }
                    } else {
                        double r2[2];
                        const bool b2 = (c >> 2) & 1u;
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const double keep = sel(b2, r4[2 * i + 1], r4[2 * i]);
                            const double send = sel(b2, r4[2 * i], r4[2 * i + 1]);
                            r2[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
                        }
                        if (s == 3) {
                            if (active) {
#pragma unroll
                                for (int i = 0; i < 2; ++i) { const int lo = 8 * i + (int)(c & 7u); blk[lo] = blk[lo] - r2[i]; }
                            }
                        } else {
                            const bool b3 = (c >> 3) & 1u;
                            const double keep = sel(b3, r2[1], r2[0]);
                            const double send = sel(b3, r2[0], r2[1]);
                            double r1 = keep + __shfl_xor_sync(0xffffffffu, send, 8);
                            if (s == 5) r1 += __shfl_xor_sync(0xffffffffu, r1, 16);
                            if (active && !(c & 16u)) { const int lo = (int)(c & 15u); blk[lo] = blk[lo] - r1; }
                        }
                    }
                }
            }
        }
        __syncthreads();
    }
}

template <int THREADS>
__device__ __forceinline__ void reduce_blocked(double* cfg0, int cfg_doubles, int off_c, int off_d1, int ng, int n,
                                               const uint16_t* mask16, const int* lvlT, int tid)
{
    reduce_blocked_rt(cfg0, cfg_doubles, off_c, off_d1, ng, n, mask16, lvlT, tid, THREADS);
}

}  // namespace cosb
