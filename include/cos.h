/*
 * include/cos.h -- C-ABI boundary of the B200-native CoS evaluation library (libcos_b200.so).
 *
 * The library evaluates, for a batch of Monte Carlo vertex configurations, the sum of the integrands
 * of ALL (cos_eval_all) or all CONNECTED (cos_eval_connected) Feynman diagrams of order n by
 * combinatorial summation (CoS):  arxiv/paper_2501_00675, Sturt & Kozik.  Citations "P:<line>" are
 * line numbers of /root/reference/PAPER.md; "R<k>" are the readings listed in DESIGN.md §4 (the
 * paper prints no formula for its graph and defers to its Ref. [10]).
 *
 * Conventions common to every call
 *   - plain C, no torch types.  Every pointer named d_* is a DEVICE pointer, every pointer named h_*
 *     is a HOST pointer; both are owned by the caller.  The library never frees, reallocates or keeps
 *     a caller pointer beyond the call, except the G0 table (borrowed until replaced/destroyed).
 *   - all floating point is IEEE FP64 (north_star; the paper itself ran FP32, reading R12), except inside the
 *     *_f32 entry points, which say so.
 *   - results are deterministic: the same call on the same inputs returns the same bits.  For n <= 10 the value of a
 *     configuration does not depend on the batch it is part of; for n >= 11 the number of configurations a thread
 *     block works on at a time follows the batch size (and is smaller for the last, partial round of a batch), and with
 *     it the order of some sums: across different batch sizes or positions in the batch the values agree to rounding
 *     (about 1e-13 relative), not bit for bit.
 *   - calls on d_* buffers are ASYNCHRONOUS on the stream given to cos_create; results are valid
 *     after the caller synchronises that stream.  Calls on h_* buffers synchronise before returning.
 *   - return value: COS_OK (0) or a negative cos_status; cos_strerror() gives the text.  No
 *     exceptions, nothing printed, no global state.  A failed call leaves outputs unspecified.
 *   - there is NO CPU fallback: every compute entry point needs a CUDA device of compute
 *     capability 10.x and fails with COS_ECUDA otherwise.
 *   - batch == 0 is legal everywhere (no work, COS_OK).  n must be in [1, COS_MAX_ORDER].
 *   - one cos_ctx must not be used from two host threads at once.
 */
#ifndef COS_B200_H
#define COS_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define COS_MAX_ORDER 16
#define COS_ABI_VERSION 1

typedef enum cos_status {
    COS_OK = 0,
    COS_EINVAL = -1,   /* bad argument: n out of range, batch < 0, NULL where not allowed, ntau < 2, ... */
    COS_ECUDA = -2,    /* CUDA runtime/driver error (no device, launch failure, ...) */
    COS_ENOMEM = -3,   /* device scratch allocation failed */
    COS_ENOTABLE = -4, /* a call that needs the G0 table was made before cos_set_g0_table */
    COS_ETOOBIG = -5   /* cos_eval_connected_noalloc: order or batch beyond the fixed capacity (COS_NOALLOC_*) */
} cos_status;

typedef struct cos_ctx cos_ctx; /* opaque; owns only internal device scratch */

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t (e.g. PyTorch's
 * torch.cuda.current_stream().cuda_stream cast to a pointer); NULL = the legacy default stream.
 * Allocates no large buffers; scratch grows on demand inside later calls.  *out receives the ctx. */
int cos_create(cos_ctx** out, int device, void* cuda_stream);

/* Free the context and its scratch (synchronises the stream first).  NULL is COS_EINVAL. */
int cos_destroy(cos_ctx* ctx);

/* Register the tabulated free propagator G0_s(x, tau) (setup step a0, not timed).
 *   spin: 0 = up, 1 = down, -1 = both species share this table.
 *   d_table: DEVICE, FP64, layout [Lx][Ly][ntau] with tau fastest; entry k holds G0 at
 *            tau_k = k*beta/(ntau-1), k = 0..ntau-1 (end points are 0+ and beta-; reading R8).
 *   The pointer is BORROWED until replaced or the ctx is destroyed.  Lx, Ly >= 1, ntau >= 2, beta > 0,
 *   Lx * Ly * ntau < 2^31 (COS_EINVAL otherwise).
 * (BASELINE.json north_star: "tabulated free propagator G0(x,tau)"; the paper takes G_ab as given.) */
int cos_set_g0_table(cos_ctx* ctx, int spin, const double* d_table, int Lx, int Ly, int ntau, double beta);

/* Step a1, G assembly for a whole batch (north_star subsystem (a)):
 *   G_s[b][i][j] = G0_s((x_i - x_j) mod L, tau_i - tau_j) by 2-point linear interpolation in tau,
 *   antiperiodic in tau:  dtau > 0: lerp(T, dtau);  dtau <= 0 and i != j: -lerp(T, dtau + beta) (R8, R9);
 *   u = dtau*(ntau-1)/beta, k = min(floor(u), ntau-2), value = fma(u-k, T[k+1]-T[k], T[k]);
 *   diagonal i == j: g_diag (equal-time convention, reading R7; default of the workloads is 0).
 *   d_xy : DEVICE int32 [batch][n][2] lattice sites, 0 <= x < Lx, 0 <= y < Ly (not range-checked)
 *   d_tau: DEVICE FP64  [batch][n], 0 <= tau < beta
 *   d_Gup, d_Gdn: DEVICE FP64 [batch][n][n] row-major outputs.  d_Gdn may be NULL or equal to d_Gup,
 *   in which case only the spin-up matrix is written (requires both species to share one table).
 * Errors: COS_ENOTABLE if a needed table is missing; COS_EINVAL for bad n/batch/NULL. */
int cos_build_G(cos_ctx* ctx, int n, long long batch, const int* d_xy, const double* d_tau,
                double g_diag, double* d_Gup, double* d_Gdn);

/* Steps a2+a3 (+a5): sum over ALL diagrams (connected and disconnected) of order n,
 *   out[b] = prod_a(-u_a) * sum_{sigma_up, sigma_dn} (-1)^{#loops} prod_i Gup[i][sigma_up(i)] Gdn[i][sigma_dn(i)]
 *          = prod_a(-u_a) * det Gup[b] * det Gdn[b],
 * computed by the layered (subset, current-vertex) graph, not by LU (top node 1, each edge
 * multiplies by one Green's function, nodes sum; -1 per closed fermion loop; R1, R6).
 *   d_Gup, d_Gdn: DEVICE FP64 [batch][n][n] row-major.  d_Gdn == d_Gup (pointer equality) means both
 *                 species share one matrix: one propagation, D = w * Z^2.
 *   d_u: DEVICE FP64 [batch][n] per-vertex couplings u_a = V_aa (reading R10), or NULL: every u_a = U.
 *   d_out: DEVICE FP64 [batch]. */
int cos_eval_all(cos_ctx* ctx, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                 const double* d_u, double U, double* d_out);

/* Steps a2+a3+a4 (+a5): the same sum restricted to CONNECTED diagrams ("all connected
 * diagrams of order n can be summed in O(n^2 2^n) operations"): the permutation pair is kept iff the
 * graph on the n vertices with edges {i,sigma_up(i)}, {i,sigma_dn(i)} is connected.  Computed as
 * propagation -> D[S] for every vertex subset -> subset recursion C[S] = D[S] - sum C[T] D[S\T]
 * (paper's Ref. [9]; north_star subsystem (c); reading R5).  Same arguments as cos_eval_all. */
int cos_eval_connected(cos_ctx* ctx, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                       const double* d_u, double U, double* d_out);

/* Whole path a1..a5 in one call: vertices in, connected value out.  G is assembled into a buffer the
 * context owns (grown on demand, freed by cos_destroy) and read back once by the evaluation kernel, i.e. the
 * call is cos_build_G + cos_eval_connected without a caller-visible G (two kernel launches on the ctx stream).
 * Both species use their registered tables; if they share one table a single propagation is done.
 * Arguments as in cos_build_G / cos_eval_connected. */
int cos_eval_connected_xt(cos_ctx* ctx, int n, long long batch, const int* d_xy, const double* d_tau,
                          double g_diag, const double* d_u, double U, double* d_out);

/* The same whole-path call with HOST buffers (pinned memory recommended): copies h_xy, h_tau (and h_u if
 * not NULL) to the device, runs a1..a5, copies the batch results back into h_out and synchronises
 * the stream before returning.  Batches of 8192 configurations or more are processed as two halves, the
 * host-to-device copy of the second half running on an internal copy stream behind the kernels of the first.  Used for end-to-end timing (h2d = batch*(8n + 8n [+ 8n]) bytes,
 * d2h = 8*batch bytes). */
int cos_eval_connected_xt_host(cos_ctx* ctx, int n, long long batch, const int* h_xy,
                               const double* h_tau, double g_diag, const double* h_u, double U,
                               double* h_out);

/* FP32 variant of steps a2..a5.  The paper runs its graph in single precision throughout
 * (Fig. 5 "FP32"; line 123: "the single-precision float value against double-precision ... on the
 * order of 10^-5 % error ... order 10 configuration"; line 125: an uplift of up to 80 % against FP64).  Same arguments,
 * layouts and return codes as cos_eval_all / cos_eval_connected (FP64 device arrays in and out): the library scales
 * the matrices of every configuration by a power of two that brings their root-mean-square entry to [1, 2) (exact;
 * the result is homogeneous of degree 2n in G, so it is multiplied by the inverse power on output -- without this
 * the products of ten small Green's functions leave the FP32 range), rounds G and u once to FP32 into buffers of its
 * own, and every later operation -- propagation, combine, connected reduction -- is FP32; the result is widened to
 * FP64 on output.  All orders 1..16 (every kernel family is instantiated for float).
 * NOTE (reading R5): this build obtains `connected` by subtracting disconnected
 * parts, so its FP32 error is about eps_32 * |D| / |C| per configuration, larger than the paper's figure, which is
 * for a subtraction-free graph; DESIGN.md reports the measured distribution. */
int cos_eval_all_f32(cos_ctx* ctx, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                     const double* d_u, double U, double* d_out);
int cos_eval_connected_f32(cos_ctx* ctx, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                           const double* d_u, double U, double* d_out);

/* On-device Monte Carlo over the vertex coordinates (reading R19).
 * (section II.B): "The integration over the vertex coordinates can then be performed by stochastic (Monte Carlo)
 * sampling"; line 137 (section IV.A): "one needs to handle proposal and acceptance of configurations ... readily
 * implemented in device-sided code"; line 87: "many Markov chain walkers".  Every configuration of the batch is an
 * independent Metropolis walker with weight |connected|.  Step t of walker w draws
 *   (r0..r3) = philox4x32_10(counter (t, 0, w_lo, w_hi), key (seed_lo, seed_hi)),  (s0..s3) = same with counter (t, 1, ..),
 * moves vertex k = r0 mod n to site (r1 mod Lx, r2 mod Ly) and time beta * u53(s0, s1), and accepts iff
 * u53(s2, s3) * |w_old| < |w_new|, with u53(a, b) = ((a << 21) ^ (b >> 11)) * 2^-53.  The proposals of all walkers
 * are evaluated by one pass of the hot path (cos_build_G + evaluation kernel), so a step is four kernel launches
 * and nothing crosses to the host.
 *   d_xy [walkers][n][2], d_tau [walkers][n]: the walkers' configurations, updated in place;
 *   d_weight [walkers]: connected value of the final configurations (out);
 *   d_accept_hist: NULL or [steps][walkers], 1 where the proposal of that step was accepted;
 *   d_accepted: NULL or [walkers] accepted proposals; d_sign_sum: NULL or [walkers], sum over the steps of the
 *   sign of the weight held after the step (numerator of the average sign).
 * Uses the table registered for both species (COS_EINVAL if two different tables are registered) and the ctx
 * loop weight.  COS_ENOTABLE without a table. */
int cos_mc_run(cos_ctx* ctx, int n, long long walkers, int steps, unsigned long long seed, int* d_xy, double* d_tau,
               double g_diag, double U, double* d_weight, unsigned char* d_accept_hist, long long* d_accepted,
               double* d_sign_sum);

/* Loop-weight generalisation (reading R17).  The paper multiplies by -1 on closing a
 * fermion loop (section IV); with N_f degenerate flavours the flavour trace of every closed loop
 * contributes a further factor N_f, so the loop factor becomes -N_f:
 *   Z_s[S] = sum_{sigma in Sym(S)} (-N_f)^{cyc(sigma)} prod_{i in S} G_s[i][sigma(i)]   (N_f = 1: (-1)^{|S|} det G_s[S,S]).
 * n_f may be any finite double (n_f = -1 turns every Z_s[S] into a permanent); it applies to every later
 * cos_eval_* call of this ctx, both species, all orders.  Default 1.  COS_EINVAL for NaN or infinity. */
int cos_set_loop_weight(cos_ctx* ctx, double n_f);

/* Half-vertex ("2n'") formulation, one species (reading R18).  The n_lines interaction
 * lines k = 0..n_lines-1 each join the half-vertices 2k and 2k+1 with the potential V_k ("interaction potentials
 * V_ab"); one species of fermion lines runs over all m = 2 n_lines half-vertices:
 *   all       = prod_k(-V_k) * sum_{sigma in S_m} (-N_f)^{cyc(sigma)} prod_i W[i][sigma(i)]
 *   connected = the same sum over the sigma whose interaction-line graph (an edge {i/2, sigma(i)/2} for every i)
 *               is connected.
 * d_W: [batch][m][m] row-major FP64, d_V: [batch][n_lines]; connected != 0 selects `connected`, else `all`;
 * d_out: [batch].  1 <= n_lines <= COS_MAX_ORDER / 2.  N_f is the ctx loop weight (cos_set_loop_weight).
 * Served by the plain one-thread-per-node kernel (propagation over the m points, D'[P] over the subsets of lines,
 * reduction over n_lines bits): correct for every size, not tuned. */
int cos_eval_halfvertex(cos_ctx* ctx, int n_lines, long long batch, const double* d_W, const double* d_V,
                        int connected, double* d_out);

/* Allocation-free evaluation of the connected sum, for callers that may not allocate device memory (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same operation and argument meaning as
 * cos_eval_connected (readings R1-R8), served by the pair
 * kernel (orders >= 11, the kernel that keeps its records in global scratch) with BOTH its record space and its item
 * descriptors in one file-scope `static __device__` array of COS_NOALLOC_SCRATCH_BYTES bytes that every GPU which
 * loads the library holds until the process exits.  The call issues kernel launches only: no cudaMalloc, cudaFree or
 * allocating library routine, and it does not touch the scratch the other entry points grow.
 *   limits : COS_NOALLOC_MIN_ORDER <= n <= COS_NOALLOC_MAX_ORDER and 0 <= batch <= COS_NOALLOC_MAX_BATCH, else
 *            COS_ETOOBIG (order or batch above the maximum) or COS_EINVAL (n below the minimum: those orders use no
 *            scratch -- call cos_eval_connected; negative batch; NULL pointers).
 *   team   : the largest team of instances per thread block, up to the one cos_eval_connected would take, whose
 *            records for a full grid fit the array; values agree with cos_eval_connected to rounding (see the
 *            determinism note above), bit for bit when the team is the same.
 *   sharing: the array is shared by EVERY call on that GPU, from any ctx and any stream, and keeps the contents of the
 *            last call.  Nothing in it has to start at zero (the descriptors are rewritten by every call, every record
 *            is written before it is read).  Two calls that overlap on the GPU (different streams or contexts) race
 *            on it and return garbage: serialise them.
 * Asynchronous on the ctx stream like the other d_* calls.  Not covered by cos_enable_kernel_timer (the timer creates
 * events on demand). */
#define COS_NOALLOC_MIN_ORDER 11
#define COS_NOALLOC_MAX_ORDER 12
#define COS_NOALLOC_MAX_BATCH (1LL << 20)
#define COS_NOALLOC_SCRATCH_BYTES (32u << 20)
int cos_eval_connected_noalloc(cos_ctx* ctx, int n, long long batch, const double* d_Gup, const double* d_Gdn,
                               const double* d_u, double U, double* d_out);

/* Cross-check switch: enable != 0 routes every later cos_eval_* call of this ctx, whatever the order, through the
 * plain one-thread-per-node kernel (the one orders 1..4 always use) instead of the tuned team / pair kernels; it
 * runs on the same device with the same arguments and is only slower.  The GPU tests use it to compare the tuned
 * kernels with a second, structurally different CUDA evaluation of SURVEY.md 8(a) a2..a5. */
int cos_debug_force_generic(cos_ctx* ctx, int enable);

/* Number of kernel launches issued by the most recent compute call on this ctx (>= 1 on success). */
int cos_last_launch_count(const cos_ctx* ctx);

/* Name of the dominant kernel variant the most recent eval call dispatched to (static string). */
const char* cos_last_kernel_name(const cos_ctx* ctx);

/* Average duration in milliseconds of the dominant (evaluation) kernel over the launches issued by
 * this ctx since the last cos_reset_kernel_timer(), measured with CUDA events recorded on the ctx
 * stream around that kernel only.  Timing is off by default (zero overhead); enable != 0 switches it
 * on.  cos_kernel_time_ms synchronises the stream.  Returns COS_EINVAL if nothing was timed. */
int cos_enable_kernel_timer(cos_ctx* ctx, int enable);
int cos_reset_kernel_timer(cos_ctx* ctx);
int cos_kernel_time_ms(cos_ctx* ctx, double* avg_ms, long long* launches);

/* Algorithmic operation count per configuration (1 FMA = 2 FLOP; no GPU needed):
 *   ext(n) = (n^2-3n+4) 2^(n-2) - 1 extend FMAs and close(n) = n 2^(n-1) close FMAs per species,
 *   2^n combine multiplies, red(n) = 3^(n-1) - 2^(n-1) reduction FMAs (connected only).
 * n_species = 1 (aliased) or 2.  Returns FLOP per configuration, or -1 for bad arguments. */
long long cos_flop_count(int n, int n_species, int connected);

/* Roofline denominators measured on the device of this ctx (synchronous, a few milliseconds each):
 *   cos_probe_dfma:  sustained FP64 FMA throughput of a register-only kernel, in TFLOP/s;
 *   cos_probe_smem:  sustained shared-memory load bandwidth (conflict-free LDS.64), in GB/s. */
int cos_probe_dfma(cos_ctx* ctx, double* tflops);
int cos_probe_smem(cos_ctx* ctx, double* gbytes_per_s);

/* Text for a status code (never NULL).  For COS_ECUDA, cos_last_cuda_error gives the CUDA text. */
const char* cos_strerror(int code);
const char* cos_last_cuda_error(const cos_ctx* ctx);

int cos_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* COS_B200_H */
