/*
 * afqmc.h -- C ABI of the B200-native batched phaseless-AFQMC local-energy library.
 *
 * What it computes (citations are to /root/reference/PAPER.md = arXiv 2209.04015, the ipie paper; letters
 * follow BASELINE.json: N orbitals, n_sigma electrons of spin sigma, Ngamma Cholesky vectors, Nw walkers):
 *
 *   for every walker w, with a single-determinant trial psi_sigma (N x n_sigma) and walker determinants
 *   phi_{sigma,w} (N x n_sigma, complex128):
 *     S_sigma      = psi_sigma^dagger phi_{sigma,w}                         PAPER.md:143  (Eq. 16)
 *     overlap      = det S_alpha * det S_beta   (returned as its logarithm)  PAPER.md:143  (Eq. 16)
 *     theta_sigma  = (phi_{sigma,w} S_sigma^-1)^T          (n_sigma x N)     PAPER.md:191  (Eq. 23), Listing 2
 *     E1           = sum_sigma sum_ip  htilde^sigma_ip theta^sigma_ip        PAPER.md:282, Eq. 2, Eq. 22
 *     T^gamma_sigma= Ltilde^gamma_sigma theta_sigma^T      (n_sigma x n_sigma)  PAPER.md:239 (Eq. 29)
 *     E            = E0 + E1 + 1/2 sum_gamma (sum_sigma Tr T^gamma_sigma)^2
 *                            - 1/2 sum_gamma sum_sigma Tr(T^gamma_sigma T^gamma_sigma)   PAPER.md:224,234 (Eq. 26, 28)
 *   where htilde_sigma = psi_sigma^dagger h and Ltilde^gamma_sigma = psi_sigma^dagger L^gamma are built once in
 *   afqmc_create (Eq. 21: "only needs to be constructed once").  T is formed and consumed on chip
 *   ("direct algorithm"); the Nw*Ngamma*n^2 tensor is never written to memory.
 *
 * Conventions common to all entry points
 *   - complex128 = two float64 (re, im) interleaved; all matrices row-major; everything little-endian.
 *   - "device" pointers are CUDA device memory of the current device; "host" pointers are ordinary (preferably
 *     pinned) host memory.  The caller owns every buffer it passes; the library reads inputs only during the
 *     call, writes only the named outputs, and owns its handle and internal workspaces until afqmc_destroy.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Return value: AFQMC_OK or a negative error code; afqmc_last_error() gives the text.  Argument errors are
 *     detected before any work is enqueued.
 *   - Tuning overrides (benchmarks only; results do not depend on them): the environment variable
 *     AFQMC_K2_PIPELINE="k,s" forces K2's shared-memory ring to s stages of k DMMA k-steps each when that fits;
 *     AFQMC_K2_SHAPE="warps,ctas_per_sm,gammas_per_tile,walkers_per_tile" forces K2's CTA shape (0 = planner's choice
 *     for the last two).  Both are read once per process.
 *   - A handle owns one set of workspaces: calls on the same handle must be ordered (one stream, or streams the
 *     caller has ordered with events); use one handle per concurrent stream.  Handles are independent of each other.
 *   - Requires compute capability 10.x (sm_100a); anything else returns AFQMC_ERR_ARCH.  There is no CPU path.
 */
#ifndef AFQMC_H_
#define AFQMC_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct afqmc_ctx afqmc_ctx; /* opaque, library-owned */

enum {
    AFQMC_OK = 0,
    AFQMC_ERR_ARG = -1,         /* null pointer, size out of range, n_walkers > max_walkers ...          */
    AFQMC_ERR_ALLOC = -2,       /* cudaMalloc failed                                                    */
    AFQMC_ERR_CUDA = -3,        /* a CUDA call or kernel launch failed                                  */
    AFQMC_ERR_ARCH = -4,        /* device is not sm_100                                                 */
    AFQMC_ERR_UNSUPPORTED = -5  /* valid input the library does not handle yet (n_sigma > 64)           */
};

#define AFQMC_MAX_NOCC 64 /* largest n_sigma supported (shared-memory inversion and register-tile limits) */

/*
 * afqmc_create -- one-time setup for a Hamiltonian and trial (Eq. 21).
 *   h1e    device, float64 [N][N], real symmetric one-body matrix h_pq (Eq. 2; used as given, no shift).
 *   chol   device, float64 [n_gamma][N][N], Cholesky vectors L^gamma_pq, each slice symmetric (Eq. 3).
 *          Not retained: may be freed after the call returns.
 *   trial  device, complex128: alpha block [N][n_alpha] followed by beta block [N][n_beta] (columns =
 *          occupied orbitals; orthonormal columns expected).  A spin block whose imaginary part is
 *          identically zero (all of BASELINE.json's configs) takes the real-Ltilde path of PAPER.md:212 (two real
 *          products per complex T); a block with a non-zero imaginary part takes the four-product path (Ltilde
 *          stored as stacked Re / Im rows), at twice the arithmetic; such a block supports n_sigma <= 52 (2 n_sigma
 *          rows must fit one K2 tile), beyond that AFQMC_ERR_UNSUPPORTED.  Non-finite entries return AFQMC_ERR_ARG.
 *   N >= 1; 0 <= n_alpha, n_beta <= min(N, AFQMC_MAX_NOCC); n_alpha + n_beta >= 1; n_gamma >= 1.
 *   e0     constant energy E0 added to every walker's energy.
 *   max_walkers >= 1 sizes the internal workspaces (theta, partial sums).
 *   The call enqueues the half-rotation on `stream` and synchronises it before returning.
 *   *out receives the handle (NULL on failure; on failure afqmc_last_error(NULL) holds the message).
 */
int afqmc_create(const double *h1e, const double *chol, const void *trial, int N, int n_alpha, int n_beta,
                 int n_gamma, double e0, int max_walkers, void *stream, afqmc_ctx **out);

/*
 * afqmc_local_energy -- the hot path: kernels K1 (overlap, determinant, inverse, theta, E1), K2 (fused exchange +
 * Coulomb traces, once per spin) and K3 (assembly), all enqueued on `stream`; returns without synchronising.
 *   walkers       device, complex128: alpha block [n_walkers][N][n_alpha] then beta block
 *                 [n_walkers][N][n_beta]  ("Nwalkers x M x N").  Need not be orthonormal.
 *   n_walkers     1 .. max_walkers.
 *   out_energies  device, complex128 [n_walkers]: local energy E_w (Eq. 26).
 *   out_overlaps  device, complex128 [n_walkers]: LOG-overlap, (re, im) = (log|<psi_T|phi_w>|, arg in (-pi, pi]).
 *   A walker exactly orthogonal to the trial (zero pivot) is data, not an error: its energy is NaN+NaN i and
 *   the real part of its log-overlap is -inf.
 *   Outputs are valid once the caller has synchronised `stream`.  No allocation, no host copy, no host sync.
 */
int afqmc_local_energy(afqmc_ctx *ctx, const void *walkers, int n_walkers, void *out_energies,
                       void *out_overlaps, void *stream);

/*
 * afqmc_local_energy_host -- the same computation with HOST buffers: copies `walkers_host` to an internal
 * device buffer, runs the kernels, copies both outputs back, and synchronises `stream` before returning.  Layouts as
 * above.  The walkers travel in three blocks -- the first eighth of the alpha block on `stream`, then the rest of it and
 * the beta block on a stream of the handle's own -- and K1 + K2 run block by block, so that all but the first copy land
 * under the kernels (results are bit-identical to afqmc_local_energy: the blocks are whole K2 column tiles).  Pinned host
 * memory makes the copies asynchronous DMA; with pageable memory they serialise.
 */
int afqmc_local_energy_host(afqmc_ctx *ctx, const void *walkers_host, int n_walkers, void *out_energies_host,
                            void *out_overlaps_host, void *stream);

/*
 * afqmc_force_bias -- copies out the Coulomb traces of the most recent afqmc_local_energy call,
 * xbar^gamma_w = sum_sigma Tr T^gamma_sigma = sum_pq G_pq L^gamma_pq   (Eq. 19, 24).
 *   out  device, complex128 [n_walkers][n_gamma], n_walkers = that of the last energy call.  Enqueued on `stream`.
 */
int afqmc_force_bias(afqmc_ctx *ctx, void *out, void *stream);

/*
 * afqmc_enable_force_bias / afqmc_force_bias_only -- the force bias WITHOUT the energy, for the propagation steps
 * between energy evaluations (25 per block in the paper's runs):
 *     xbar^gamma_w = sum_sigma sum_ip Ltilde^gamma_ip theta_ip           PAPER.md:195 (Eq. 24), Listing 3
 * i.e. one real GEMM [Ngamma x n N] . [n N x 2 Nw] per spin (re and im planes of theta as columns) on the FP64 tensor
 * cores, after K1 has built theta.
 *   afqmc_enable_force_bias builds a second copy of Ltilde in that GEMM's operand order (about the size of the first:
 *   Ngamma * n * N doubles per spin, twice that for a complex trial block) from `chol` (device, the array given to
 *   afqmc_create, not retained) and synchronises `stream`.  Idempotent.
 *   afqmc_force_bias_only enqueues K1, the GEMM (one launch per spin) and a combine kernel on `stream`:
 *     walkers  device, layout as in afqmc_local_energy;  n_walkers 1 .. max_walkers
 *     out      device, complex128 [n_walkers][n_gamma]
 *   Returns AFQMC_ERR_ARG if afqmc_enable_force_bias has not been called on this handle.
 */
int afqmc_enable_force_bias(afqmc_ctx *ctx, const double *chol, void *stream);
int afqmc_force_bias_only(afqmc_ctx *ctx, const void *walkers, int n_walkers, void *out, void *stream);

/*
 * afqmc_spin_squared -- a second mixed estimator from the same half-rotated Green's function (Eq. 31
 * with the index order of Listing 6):
 *     s2_w = <psi_T|S^2|phi_w> / <psi_T|phi_w> = n_beta + M_S (M_S + 1) - sum_pq G^alpha_pq G^beta_qp ,   M_S = (n_alpha - n_beta) / 2
 * for the walkers of the most recent afqmc_local_energy / afqmc_force_bias_only call (it reads the theta those calls
 * left in the handle).  out: device, complex128 [n_walkers of that call].  Enqueued on `stream`.
 */
int afqmc_spin_squared(afqmc_ctx *ctx, void *out, void *stream);

/*
 * afqmc_greens_function -- optional full one-body Green's function of one spin sector, for user-written mixed
 * estimators (the paper's greens_function(walkers, trial, build_full=True)):
 *     G^sigma_pq = <psi_T|a+_p a_q|phi_w> / <psi_T|phi_w> = [phi S^-1 psi^dagger]_qp = sum_j theta^sigma_jq conj(psi^sigma_pj)
 *                                                                                      PAPER.md:174, 187 (Eq. 20, 22)
 * for the walkers of the most recent afqmc_local_energy / afqmc_force_bias_only call.
 *   spin  0 = alpha, 1 = beta.   out: device, complex128 [n_walkers of that call][N][N], row-major in (p, q);
 *   n_walkers * N * N * 16 bytes (344 MB per spin at N = 290, 256 walkers).  Enqueued on `stream`.
 */
int afqmc_greens_function(afqmc_ctx *ctx, int spin, void *out, void *stream);

/*
 * afqmc_phaseless_weights -- the weight update of the hybrid phaseless propagation (Eq. 7, 8, 10-12),
 * for a caller that applies its own propagator B(x - xbar) to the walkers and evaluates the overlaps before and after
 * with afqmc_local_energy / afqmc_force_bias_only:
 *     O = exp(log_ovlp_new - log_ovlp_old),   I = O exp(x . xbar - xbar . xbar / 2),   w_new = |I| max(0, cos(arg O)) w
 *   x             device, float64 [n_walkers][n_gamma]      auxiliary fields drawn by the caller (Eq. 4)
 *   xbar          device, complex128 [n_walkers][n_gamma]   the shift of Eq. 9, xbar = -sqrt(dt) <v'>.  NOT the output
 *                 of afqmc_force_bias[_only], which is Eq. 19's sum_pq G_pq L^g_pq: with the propagator of
 *                 afqmc_propagate (v' = i v) the two are related by xbar = -i sqrt(dt) * (Eq. 19)
 *   log_ovlp_old/new  device, complex128 [n_walkers]        (log|ovlp|, arg ovlp) as returned in out_overlaps
 *   weights_in/out    device, float64 [n_walkers]           may alias
 * No handle: the call keeps no state.  Enqueued on `stream`.
 */
int afqmc_phaseless_weights(int n_walkers, int n_gamma, const double *x, const void *xbar, const void *log_ovlp_old,
                            const void *log_ovlp_new, const double *weights_in, double *weights_out, void *stream);

/*
 * afqmc_sample_fields -- the auxiliary fields of one propagation step, x[w][gamma] ~ N(0, 1) (Eq. 4: "p(x) is
 * the normal distribution").  The paper names no generator; this is a counter-based one (Philox4x32-10 + Box-Muller,
 * DESIGN.md section 3 row 21; csrc/k10_fields.cuh states the exact mapping), so the call keeps no state:
 *     x[w][2b], x[w][2b+1]  <-  Philox4x32-10(counter = (b, first_walker + w, step lo, step hi), key = (seed lo, seed hi))
 * A walker's fields depend only on (seed, step, its global index first_walker + w, gamma): not on the batch, the rank or
 * the launch.  Optional: afqmc_propagate takes x from any source.
 *   x   device, float64 [n_walkers][n_gamma].   n_walkers, n_gamma >= 1, first_walker >= 0.   Enqueued on `stream`.
 */
int afqmc_sample_fields(unsigned long long seed, unsigned long long step, int first_walker, int n_walkers, int n_gamma,
                        double *x, void *stream);

/*
 * afqmc_enable_propagation / afqmc_propagate -- one step of the hybrid phaseless propagation for all walkers
 * (Eq. 6-13), the other hotspot next to the local energy.
 *
 * The paper defines the propagator only through Eq. 4, exp(-dt H) = int dx p(x) B(x) + O(dt^2) with p the normal
 * distribution.  The reading built here (the oracle pins it with Eq. 4 itself):
 *     h'       = h - 1/2 sum_g L^g L^g          Eq. 2 is normal ordered: H = sum h'_pq a+_p a_q + 1/2 sum_g v_g^2,
 *                                               v_g = sum_pr L^g_pr a+_p a_r  (Eq. 2, 3)
 *     B(dt, y) = exp(-dt h'/2) exp(i sqrt(dt) sum_g y_g L^g) exp(-dt h'/2)     acting on both spin blocks (Eq. 4)
 *     xbar_g   = -i sqrt(dt) sum_pq G_pq L^g_pq                                Eq. 9 with v' = i v; the sum is Eq. 19
 *     phi'     = B(dt, x - xbar) phi                                           Eq. 13
 *     O        = <psi_T|phi'> / <psi_T|phi>                                    Eq. 8
 *     w'       = |O exp(x.xbar - xbar.xbar/2)| max(0, cos(arg O)) w            Eq. 7, 10-12
 * No mean-field shift, no population control, no re-orthonormalisation (the paper does not describe them).
 *
 * afqmc_enable_propagation(ctx, h1e, chol, dt, stream): one-time setup for time step dt > 0 (fixed per handle).
 *   h1e, chol   device, the arrays given to afqmc_create (not retained).
 *   Builds h', exp(-dt h'/2) (scaling and squaring, on the GPU), a third packing of the Cholesky vectors
 *   (upper triangles only, n_gamma * N (N + 1) / 2 doubles: every L^g is symmetric) as the operand of the field GEMM, the force-bias operand (afqmc_enable_force_bias) and
 *   work buffers (3 * max_walkers * N^2 doubles for the per-walker matrices sum_g y_g L^g, among others).
 *   Synchronises `stream`.  A second call on the same handle returns AFQMC_ERR_ARG.
 *
 * afqmc_propagate(ctx, walkers, n_walkers, x, weights_in, weights_out, log_ovlp_out, taylor_order, stream):
 *   walkers       device, complex128, layout of afqmc_local_energy; READ AND OVERWRITTEN with phi' (Eq. 13).
 *   x             device, float64 [n_walkers][n_gamma]: the auxiliary fields, drawn by the caller from the standard
 *                 normal distribution (Eq. 4).  The library draws no random numbers.
 *   weights_in / weights_out   device, float64 [n_walkers]; may alias.
 *   log_ovlp_out  device, complex128 [n_walkers] or NULL: (log|<psi_T|phi'>|, arg) of the propagated walkers.
 *   taylor_order  0 .. 64: exp(A) phi is evaluated as sum_{k <= order} A^k phi / k!  (A = i sqrt(dt) sum y_g L^g).  The
 *                 truncation error, about ||A||^(order+1) / (order+1)!, is the caller's to bound; the paper does not
 *                 state an order (6 is customary for dt ~ 0.005 and molecular Hamiltonians).
 *   Kernels, all on `stream`, no host synchronisation: K1 (theta, overlap of phi), force-bias GEMM, field GEMM
 *   [N(N+1)/2 x n_gamma].[n_gamma x 2 n_walkers] on the FP64 tensor cores, order + 2 batched [N x N].[N x 2(n_alpha+n_beta)]
 *   products (the series by Horner's rule), K1 again (overlap of phi'), weight update.  A walker orthogonal to the trial before or after the step gets
 *   weight NaN (its log-overlap is -inf).  Afterwards the handle's theta belongs to phi' (afqmc_spin_squared,
 *   afqmc_greens_function refer to the propagated walkers; afqmc_force_bias has nothing to return).
 *
 * afqmc_propagation_xbar: copies out the xbar (Eq. 9) of the last afqmc_propagate call, complex128 [n_walkers][n_gamma].
 * afqmc_propagate_phase_ms: with afqmc_set_profiling(ctx, 1), device times of the last afqmc_propagate call:
 *   ms[0] K1 + overlap, [1] force-bias GEMM, [2] fields + field GEMM, [3] one-body and Taylor products, [4] K1 + weights.
 */
int afqmc_enable_propagation(afqmc_ctx *ctx, const double *h1e, const double *chol, double dt, void *stream);
int afqmc_propagate(afqmc_ctx *ctx, void *walkers, int n_walkers, const double *x, const double *weights_in,
                    double *weights_out, void *log_ovlp_out, int taylor_order, void *stream);
int afqmc_propagation_xbar(afqmc_ctx *ctx, void *out, void *stream);
int afqmc_propagate_phase_ms(afqmc_ctx *ctx, float ms[5]);

/*
 * afqmc_log_overlap_static -- the log-overlaps alone, from an entry point that ALLOCATES NOTHING: no handle, no cudaMalloc /
 * cudaFree, no allocating library routine, no host synchronisation.  For callers that cannot allocate: code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it.
 *     out_overlaps[w] = (log|<psi_T|phi_w>|, arg <psi_T|phi_w>),   <psi_T|phi_w> = det(psi_alpha^dagger phi_alpha,w) det(psi_beta^dagger phi_beta,w)
 *                                                                                   PAPER.md:143 (Eq. 16), 146-150
 * computed by kernel K1 as afqmc_local_energy runs it (same values as that call's out_overlaps).  Its scratch -- the trial
 * packed for the tensor cores, the theta K1 writes as a by-product, per-walker partial results -- lives in ONE file-scope
 * device array of AFQMC_STATIC_SCRATCH_BYTES that every GPU holds from the moment it loads the library until the process
 * exits.  Sizes that need more return AFQMC_ERR_UNSUPPORTED with the byte counts in the message:
 *     8 n_max N + 16 sum_sigma N n_sigma + 16 n_walkers sum_sigma N n_sigma (+ padding to tiles of 8 / 4 / 32) + 64 n_walkers  bytes,
 * e.g. N = 290, n_alpha = n_beta = 26: up to 62 walkers per call; N = 100, n = 20: up to 260; N = 500, n = 50: up to 18.
 *   trial         device, complex128, layout of afqmc_create (read on every call: no state is kept between calls)
 *   walkers       device, complex128, layout of afqmc_local_energy;  n_walkers >= 1
 *   out_overlaps  device, complex128 [n_walkers]
 * Enqueued on `stream`, returns without synchronising.  ALL calls, from all threads and streams, share the one array (it
 * keeps the last call's contents; the call clears what must start at zero): calls that overlap on the GPU -- different
 * streams without an ordering between them -- race.  Order them, or use handles (afqmc_create) instead.
 */
#define AFQMC_STATIC_SCRATCH_BYTES 16777216 /* 16 MiB per GPU that loads the library */
int afqmc_log_overlap_static(const void *trial, const void *walkers, int N, int n_alpha, int n_beta, int n_walkers,
                             void *out_overlaps, void *stream);

/* Frees the handle and every internal buffer.  NULL is allowed. */
void afqmc_destroy(afqmc_ctx *ctx);

/* Message of the last error on this handle (or of the last failed afqmc_create when ctx == NULL).
 * Library-owned, valid until the next call on the same handle; never freed by the caller. */
const char *afqmc_last_error(const afqmc_ctx *ctx);

/* ---- introspection used by the benchmark and the tests (no effect on results) ------------------------- */

typedef struct afqmc_info {
    int N, n_alpha, n_beta, n_gamma, max_walkers;
    int k_steps;           /* ceil(N/4): DMMA k-steps per output tile                                   */
    int tile_rows[2];      /* per spin: rows (gamma,i) of the K2 CTA tile, multiple of 8                 */
    int tile_cols[2];      /* per spin: real columns (plane,walker,j) of the K2 CTA tile, multiple of 8  */
    int gammas_per_tile[2];
    int walkers_per_tile[2];
    int warps_m[2], mt[2], nt[2], stages[2], ksteps_per_chunk[2];
    int k2_smem_bytes[2];
    long long ltilde_bytes;   /* packed half-rotated Cholesky tensor, both spins, including padding      */
    long long theta_bytes;    /* packed theta planes for max_walkers, both spins, including padding      */
    long long kernel_launches; /* kernels launched by this handle so far (create + energy calls)         */
} afqmc_info;

int afqmc_get_info(const afqmc_ctx *ctx, afqmc_info *info);

/* afqmc_plan -- host only (no CUDA call, works without a GPU): the K2 tile shape, pipeline depth and packed
 * operand sizes afqmc_create would choose for these sizes (kernel_launches = 0).  Same argument checks and
 * error codes as afqmc_create. */
int afqmc_plan(int N, int n_alpha, int n_beta, int n_gamma, int max_walkers, afqmc_info *info);
/* afqmc_plan_trial -- the same for a trial whose alpha / beta block is complex (complex_alpha / complex_beta != 0:
 * the four-product path, 2 n_sigma rows per gamma block); afqmc_plan is the all-real case. */
int afqmc_plan_trial(int N, int n_alpha, int n_beta, int n_gamma, int max_walkers, int complex_alpha, int complex_beta,
                     afqmc_info *info);

/* Per-kernel device times of energy calls.  enable != 0 makes every later afqmc_local_energy record CUDA
 * events around K1, K2 (both spins) and K3 on the caller's stream. */
int afqmc_set_profiling(afqmc_ctx *ctx, int enable);
/* After the stream has been synchronised: ms[0..2] = K1, K2 (both spins), K3 of the most recent profiled call. */
int afqmc_last_kernel_ms(afqmc_ctx *ctx, float ms[3]);
/* Mean of the same three times over the profiled calls since afqmc_set_profiling(ctx, 1) (the most recent
 * 256 at most); *n_calls = how many were averaged.  The stream must have been synchronised. */
int afqmc_mean_kernel_ms(afqmc_ctx *ctx, float ms[3], int *n_calls);

/*
 * afqmc_fp64_peak -- register-resident FP64 throughput microbenchmark used as the roofline denominator
 * (MEASURED_PEAKS.json has no FP64 entry).  mode 0: DMMA.8x8x4 (mma.sync m8n8k4 f64) chains;
 * mode 1: DFMA chains.  Runs `launches` back-to-back launches on `stream`, synchronises, and writes the
 * achieved TFLOP/s of the whole sequence to *tflops.
 */
int afqmc_fp64_peak(int mode, int launches, double *tflops, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* AFQMC_H_ */
