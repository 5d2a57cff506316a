/*
 * cheb_dm.h -- C ABI of the B200-native dense Chebyshev Fermi-operator solver.
 *
 * Hot path of arXiv 2306.12616 ("A fast, dense Chebyshev solver for electronic structure on
 * GPUs"), cited below as PAPER.md:<line>:
 *
 *     D = f(H) = [I + exp(beta (H - mu I))]^{-1}                         (Eq. 3)
 *       ~ sum_{n=0}^{M-1} c_n T_n(X),   X = (2H - (a+b) I)/(b - a)
 *
 * evaluated with the baby-step/giant-step factorisation of Eq. (4):
 * T_2..T_k by T_{a+b} = 2 T_a T_b - T_|a-b| (Eq. 7, 22-23, Algorithm 1),
 * then p-1 further products in T_k whose epilogues add the independent low-order sums of
 * Eq. (21).  k*p >= M; M is the number of terms (the paper's L+1), p is the
 * paper's `m`.
 *
 * Conventions
 *  - Every call returns a cheb_dm_status_t (0 = OK); nothing throws or aborts; on error no
 *    output argument is written.
 *  - "device pointer" = CUDA global memory of the device that was current in cheb_dm_plan();
 *    "host pointer" = ordinary host memory.  Matrices are dense row-major FP64; DEVICE matrices H and D
 *    have the leading dimensions of the plan options ldh / ldd (default N: row i starts at element
 *    i*N), HOST matrices always have leading dimension N.  H must be symmetric (row-major == col-major).
 *  - Batched calls (cheb_dm_*_batch: many independent small Hamiltonians) take HOST
 *    arrays of nbatch device (or host) matrix pointers, nbatch <= the plan option max_batch; matrix s of
 *    the batch lives in "slot" s of the plan's workspace.  The single-matrix calls are the nbatch = 1 case.
 *  - The plan owns its workspace (cudaMalloc'ed in cheb_dm_plan(), freed in cheb_dm_destroy());
 *    the caller owns H, D and every output buffer.  D must not alias H.
 *  - cheb_dm_compute[_batch] / cheb_dm_solve[_batch] (mu_out == NULL) / cheb_dm_assemble / cheb_dm_trace[_batch] /
 *    cheb_dm_moments (tau_host == NULL) / cheb_dm_product are asynchronous on the given stream (a
 *    cudaStream_t passed as void*; NULL = legacy default stream), allocate nothing, read no environment
 *    variable, never synchronise with the host and may be captured into a CUDA graph.  Calls that
 *    return scalars to HOST memory (cheb_dm_get_bounds, cheb_dm_get_scalars, cheb_dm_get_coeffs,
 *    cheb_dm_solve_mu, cheb_dm_get_T, cheb_dm_check) synchronise the stream they are given.
 *  - Errors the DEVICE detects (non-finite bounds, the stability guard of the power-basis recursion, a
 *    dependency watchdog) are sticky flags: they survive later computes on the plan and are reported -- and
 *    cleared -- by the next cheb_dm_check / cheb_dm_wait / cheb_dm_compute_host.
 *  - A plan is not thread-safe; distinct plans are independent.  There is no CPU fallback: without
 *    a CUDA device cheb_dm_plan() returns CHEB_DM_ECUDA.
 */
#ifndef CHEB_DM_H
#define CHEB_DM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cheb_dm_plan_s* cheb_dm_plan_t; /* opaque, owned by the library */

typedef enum { CHEB_DM_F64 = 0 } cheb_dm_dtype_t; /* the paper and all configs are FP64 */

typedef enum {
    CHEB_DM_OK = 0,
    CHEB_DM_EINVAL = 1,       /* bad argument (N < 1, M < 1, NULL pointer, bad option)          */
    CHEB_DM_EALLOC = 2,       /* workspace allocation failed                                     */
    CHEB_DM_ECUDA = 3,        /* CUDA runtime/driver error, or no device                         */
    CHEB_DM_ESTATE = 4,       /* call order: compute before coeffs, solve_mu before moments ...  */
    CHEB_DM_EBOUNDS = 5,      /* b <= a or non-finite bounds                                     */
    CHEB_DM_EUNSUPPORTED = 6, /* dtype other than CHEB_DM_F64                                    */
    CHEB_DM_ENOCONV = 7,      /* stability guard of the power-basis outer recursion (Eq. 4): the table d
                                 computed on the device has max|d| 2^-52 p > 1e-12 (d grows like 2^p, Eq. 12,
                                 PAPER.md:136; reading A6); D was still written but may have lost
                                 accuracy.  Reported by cheb_dm_check / cheb_dm_wait / cheb_dm_compute_host. */
    CHEB_DM_ESIZE = 8         /* cheb_dm_bounds_static: N beyond CHEB_DM_STATIC_MAX_N (the fixed device scratch)   */
} cheb_dm_status_t;

/* Outer (giant-step) recursion.
 *  CHEB_DM_OUTER_CHEBYSHEV (default): Clenshaw recursion in T_k,
 *      B_l = G_l + 2 T_k B_{l+1} - B_{l+2},  D = G_0 + T_k B_1 - B_2,  G_l = sum_i g_{i,l} T_i,
 *      with g_{i,l} = d_i^T a_l the intermediate of Eq. (16)-(17).  Same p-1
 *      products and the same independent low-order sums as Eq. (4); stable in FP64.
 *  CHEB_DM_OUTER_POWER: Eq. (4) literally, acc <- S_j + T_k acc with S_j = sum_i d_{i,j} T_i
 *      (Eq. 21).  d grows like 2^p; reading A6.                  */
typedef enum { CHEB_DM_OUTER_CHEBYSHEV = 0, CHEB_DM_OUTER_POWER = 1 } cheb_dm_outer_t;

/* Scheduling of the products.
 *  CHEB_DM_SCHED_GROUPED (default): one persistent kernel runs every product of the solve; the
 *      independent baby-step products of a stage (Algorithm 1) run concurrently
 *      and successive giant steps are pipelined at column-panel granularity.
 *  CHEB_DM_SCHED_SERIAL: one launch per product on the stream (the paper's single-stream mode,
 *      PAPER.md:190); used as the ablation baseline.                                            */
typedef enum { CHEB_DM_SCHED_GROUPED = 0, CHEB_DM_SCHED_SERIAL = 1 } cheb_dm_sched_t;

/* Operand pairing of the baby steps (any a+b=n is valid by Eq. 7).
 *  CHEB_DM_PAIR_AUTO (default) = CHEB_DM_PAIR_BALANCED.
 *  CHEB_DM_PAIR_ALG1: Algorithm 1's pairing, ceil(log2 k) stages.
 *  CHEB_DM_PAIR_SERIAL: T_{n+1} = 2 T_1 T_n - T_{n-1} (k-1 serial products; best rounding).
 *  CHEB_DM_PAIR_BALANCED: T_n = 2 T_ceil(n/2) T_floor(n/2) - T_{0 or 1}: same stages, concurrency and cost as
 *      Algorithm 1, no long chains through T_{2^j} unless n is a power of two.  On spectra concentrated at
 *      x~ = 0 (cfg4) Algorithm 1's squaring chains leave |dtr D| = 7.7e-10 of the 1e-9 gate, the balanced
 *      pairing 1.3e-12 (reading A7b), hence the default.                                          */
typedef enum { CHEB_DM_PAIR_AUTO = 0, CHEB_DM_PAIR_SERIAL = 1, CHEB_DM_PAIR_BALANCED = 2, CHEB_DM_PAIR_ALG1 = 3 } cheb_dm_pairing_t;

typedef struct {
    int k;       /* baby-step block size; 0 = auto: ceil(sqrt(M))                 */
    int p;       /* number of Horner blocks (paper's m); 0 = auto: ceil(M/k); need k*p >= M     */
    int outer;   /* cheb_dm_outer_t                                                              */
    int sched;   /* cheb_dm_sched_t                                                              */
    int pairing; /* cheb_dm_pairing_t                                                            */
    int tile;    /* CTA tile (warp tile): 0 = auto, 1 = 128x128 (32x32), 2 = 128x64 (32x32), 3 = 64x64 (32x32),
                    4 = 64x32 (16x16), 5 = 64x32 (32x16), 6 = 128x64 (32x16), 7 = 32x32 (16x16, 2 CTAs/SM), 8 = 112x64 (16x32),
                    9 = 64x64 (32x16), 10 = 64x32 (16x16, 2 CTAs/SM); 11 = 64x32 and 12 = 64x64 in the kernel with specialised
                    epilogue warps (the consumer warps park a finished tile in shared memory and start the next item while
                    four epilogue warps combine, store, mirror and publish it).  auto: 11 or 12 for N >= 450 (whichever needs
                    fewer whole waves x tile area per product level on this device), 4 or 7 below               */
    int fuse_sums; /* low-order sums G_l / S_j of Eq. (21).  0 = auto; 1 = formed inside the
                      giant-step epilogues from T_1..T_{k-1} (no extra workspace; p(k-1) N^2 8 bytes of reads per
                      solve, L2 hits while the baby block fits L2); 2 = all p sums formed in one batched pass
                      (form_sums_dmma_kernel, a skinny GEMM on the tensor cores: each T_i read ceil(p/16) times, p extra workspace matrices), the
                      epilogues then add one tile.  auto = 2 when k N^2 8 B > 96 MiB.  With the resident giant-step
                      kernel (giant = 2) the sums are always formed inside that kernel by the CTA that consumes
                      them (reported as 2).  No mode makes the per-term AXPY passes of PAPER.md:234.          */
    int giant;   /* giant steps at N <= 512: 0 = auto, 1 = generic grouped kernel, 2 = resident-multiplier kernel (each
                    CTA keeps its 32 rows of T_k in shared memory for all p-1 products and runs two column
                    panels as independent chains; needs tile 4, 5 or 7 and grouped scheduling, else falls back; a plan with
                    max_batch > 1 whose batches gather the sums in the epilogues (fuse_sums = 1) runs its single solves in the
                    generic kernel as well: reported as 1) */
    int symmetric; /* symmetric-tile skipping: 0 = auto (on), 1 = off, 2 = on.  Every matrix of the solve is a polynomial
                    of X, hence symmetric (the paper's magma_dgemm does not use this): only the tiles of a
                    product that touch the lower triangle are computed, each mirrors its 8x8 blocks into the skipped
                    tiles (transposed in registers, stored row-contiguously).  ~45 % fewer tensor flops per product;
                    cheb_dm_flops_per_compute counts only the executed tiles.  H must be symmetric either way.        */
    int max_batch; /* matrices per grouped launch (cheb_dm_compute_batch): 0 or 1 = single solves only,
                      at most 64.  The workspace holds max_batch slots; with max_batch > 1 the tile shape is chosen for
                      the batch and batched giant steps run in the generic grouped kernel.                          */
    int ldh;       /* leading dimension (elements) of the caller's DEVICE matrices H; 0 = N; must be >= N.          */
    int ldd;       /* the same for the DEVICE output matrices D.                                                  */
    int moments;   /* 0 = auto (on), 1 = off, 2 = on: keep the giant block U_j = T_{jk}(X), j = 2..p-1, in the workspace
                      (p - 2 more matrices per slot, + p for the low-order sums) -- needed by cheb_dm_moments,
                      cheb_dm_solve and cheb_dm_assemble (EUNSUPPORTED when off).                                   */
    int host_slots; /* staging sets of the host entry points allocated at plan time: 0 = none (the first host call
                      allocates what it needs -- the one exception to "compute calls allocate nothing"), 1 = one
                      (cheb_dm_compute_host), 2 = both + copy streams/events (cheb_dm_compute_host_async).         */
    int sliced;     /* digits S of cheb_dm_product_sliced: 0 = off, 2..8: the plan allocates the int8 digit
                      planes of two operands (2 S N kpad bytes, kpad = N rounded up to 64) and their scale vectors.        */
    int sliced_solve; /* 1: every product of the plan (baby steps, giant steps, and the giant block of cheb_dm_moments /
                      cheb_dm_solve) runs on the sliced int8 tensor path (sliced digits, default 8) instead of the FP64 DMMA
                      kernel: one launch per product, each result sliced once, k + 5 (+ p - 2 with moments) digit sets in the
                      workspace; single solves only (max_batch <= 1), low-order sums pre-formed; cheb_dm_solve / assemble then
                      assemble D with the nested giant steps instead of the long-K product.  Pays from N ~ 2000 (DESIGN.md
                      section 6). */
} cheb_dm_options_t;

/* Create a plan for N x N matrices and an M_terms-term expansion.  Chooses (k,p), allocates the
 * workspace (per slot k+3 padded matrices, + p when the low-order sums are parked, + p-2 for the giant block, + scalar tables) and builds the
 * product/tile/dependency tables.
 * plan: host pointer, receives the handle.  EINVAL: N<1, M_terms<1, k*p<M; EUNSUPPORTED: dtype. */
cheb_dm_status_t cheb_dm_plan(cheb_dm_plan_t* plan, int N, int M_terms, cheb_dm_dtype_t dtype);
/* Same with explicit options (host pointer; NULL = defaults). */
cheb_dm_status_t cheb_dm_plan_ex(cheb_dm_plan_t* plan, int N, int M_terms, cheb_dm_dtype_t dtype,
                                 const cheb_dm_options_t* opts);
cheb_dm_status_t cheb_dm_destroy(cheb_dm_plan_t plan);

/* Set the Fermi function and the spectral bounds used by the next cheb_dm_compute().
 * beta: inverse temperature (>0, finite); mu: chemical potential (Eq. 2-3).
 * bounds: host pointer to {a, b} = (eps_a, eps_b) of PAPER.md:96, or NULL => Gershgorin bounds
 *   a = min_i(h_ii - R_i), b = max_i(h_ii + R_i), R_i = sum_{j!=i}|h_ij|, computed from H on the
 *   device at compute time (a == b is widened to [a-1, b+1]).
 * The Chebyshev coefficients c_n (n < M) of f~(x) = 1/(1+exp(beta~ (x - mu~))),
 *   beta~ = beta (b-a)/2, mu~ = (2 mu - (a+b))/(b-a), are computed ON THE DEVICE inside
 *   cheb_dm_compute() by the DCT at the N_q = 2^ceil(log2(4M)) Chebyshev nodes
 *   x_j = cos(pi (j+1/2)/N_q):  c_n = ((2 - delta_n0)/N_q) sum_j f~(x_j) cos(n pi (j+1/2)/N_q)
 *   (c_0 not halved: the expansion is sum c_n T_n), followed by the tables g (and d)
 *   of Eq. (16)-(20).
 * EINVAL: non-finite beta/mu or beta <= 0; EBOUNDS: explicit bounds with b <= a or non-finite. */
cheb_dm_status_t cheb_dm_coeffs(cheb_dm_plan_t plan, double beta, double mu, const double* bounds);

/* D <- sum_{n<M} c_n T_n(X) for the symmetric H (Eq. 3-4).  dH, dD: device pointers, N rows of N doubles,
 * leading dimensions ldh / ldd (plan options; default N).  Runs, on `cuda_stream` and without host synchronisation: bounds (Gershgorin
 * unless explicit) + rescale of H into X; coefficient tables; baby steps T_2..T_k; giant steps.
 * ESTATE if cheb_dm_coeffs() was never called; EINVAL on NULL/aliased pointers. */
cheb_dm_status_t cheb_dm_compute(cheb_dm_plan_t plan, const double* dH, double* dD, void* cuda_stream);

/* Batched form (SURVEY 8(f)-2; the many-small-Hamiltonians use case of PAPER.md:35, :55): nbatch independent
 * solves, D_s <- sum c_n(mu_s) T_n(X_s), in ONE set of grouped launches: one front-end launch over all matrices
 * (each with its own Gershgorin bounds and coefficient tables), one persistent baby-step launch and one
 * giant-step launch whose work lists are the union over the batch, claimed level by level and matrix by
 * matrix, so that the independent products of different matrices fill the SMs and hide one another's serial
 * chain.  dH, dD: HOST arrays of nbatch device pointers (matrices as in cheb_dm_compute); mu: HOST array of
 * nbatch chemical potentials, or NULL = the mu of cheb_dm_coeffs for all; beta and the bounds mode are those of
 * cheb_dm_coeffs.  EINVAL: nbatch < 1 or > max_batch, NULL / aliased pointers, non-finite mu. */
cheb_dm_status_t cheb_dm_compute_batch(cheb_dm_plan_t plan, int nbatch, const double* const* dH, double* const* dD,
                                       const double* mu, void* cuda_stream);

/* Host-buffer form of cheb_dm_compute (+ cheb_dm_trace): the end-to-end call a user without device
 * memory makes.  hH, hD: HOST pointers, N*N doubles (ld N), pinned memory recommended; h_trace: HOST pointer
 * to 1 double, or NULL.  On `cuda_stream`: copies H to a plan-owned device buffer, runs cheb_dm_compute,
 * the trace kernel, copies D (and tr D) back and SYNCHRONISES the stream before returning, so hD is
 * valid on return.  Same errors as cheb_dm_compute. */
cheb_dm_status_t cheb_dm_compute_host(cheb_dm_plan_t plan, const double* hH, double* hD, double* h_trace,
                                      void* cuda_stream);

/* Pipelined form of cheb_dm_compute_host for a batch of solves on one plan: returns as soon as the work is queued.
 * The H2D copy of call n+1 and the D2H copies of call n-1 run on two plan-owned copy streams and overlap the kernels
 * of call n (two device staging slots; the kernels themselves run on `cuda_stream` in call order).  hH must stay
 * valid and hD / h_trace must not be read until cheb_dm_wait() returns; pinned host memory is needed for the copies
 * to be asynchronous.  The Fermi parameters are those of the last cheb_dm_coeffs() at the time of the call.
 * cheb_dm_wait: waits for every queued call and performs cheb_dm_check(). */
cheb_dm_status_t cheb_dm_compute_host_async(cheb_dm_plan_t plan, const double* hH, double* hD, double* h_trace,
                                            void* cuda_stream);
cheb_dm_status_t cheb_dm_wait(cheb_dm_plan_t plan, void* cuda_stream);
/* Batched host forms: hH, hD HOST arrays of nbatch HOST matrix pointers (N*N doubles each, ld N, pinned
 * recommended); h_trace: HOST pointer to nbatch doubles or NULL; mu as in cheb_dm_compute_batch.  The _async form
 * queues the batch (pipelined over two staging sets like cheb_dm_compute_host_async; results valid after
 * cheb_dm_wait), the other synchronises and checks before it returns. */
cheb_dm_status_t cheb_dm_compute_batch_host(cheb_dm_plan_t plan, int nbatch, const double* const* hH, double* const* hD,
                                            double* h_trace, const double* mu, void* cuda_stream);
cheb_dm_status_t cheb_dm_compute_batch_host_async(cheb_dm_plan_t plan, int nbatch, const double* const* hH,
                                                  double* const* hD, double* h_trace, const double* mu, void* cuda_stream);

/* trace_out[0] <- tr D = sum_i D_ii (electron count, north_star item 4).  dD: device pointer (N*N,
 * ld N).  trace_out: DEVICE pointer (or pinned mapped host memory), 1 double, written
 * asynchronously on the stream in a fixed summation order (bitwise reproducible). */
cheb_dm_status_t cheb_dm_trace(cheb_dm_plan_t plan, const double* dD, double* trace_out, void* cuda_stream);

/* Batched trace: trace_out[s] <- tr D_s, s < nbatch (dD: HOST array of device pointers, ld = option ldd;
 * trace_out: DEVICE pointer to nbatch doubles), one launch. */
cheb_dm_status_t cheb_dm_trace_batch(cheb_dm_plan_t plan, int nbatch, const double* const* dD, double* trace_out,
                                     void* cuda_stream);

/* Bounds {a,b} used by the last cheb_dm_compute()/cheb_dm_moments() (host pointer, 2 doubles).
 * Synchronises `cuda_stream`.  EBOUNDS if the device flagged non-finite bounds. */
cheb_dm_status_t cheb_dm_get_bounds(cheb_dm_plan_t plan, double* bounds_out, void* cuda_stream);

/* Device-side scalars of slot `slot` (< max_batch) after the last call: out[0..3] = {a, b, mu, N_e(mu)} (host
 * pointer; N_e is set by the bisection only).  Synchronises `cuda_stream`.  EBOUNDS as cheb_dm_get_bounds. */
cheb_dm_status_t cheb_dm_get_scalars(cheb_dm_plan_t plan, int slot, double* out4, void* cuda_stream);

/* Scalar tables of the last compute, copied to host memory (any pointer may be NULL):
 *   c_out[k*p]  c_n (zero for n >= M);   g_out[k*p]  g_{i,l} at [i*p + l];
 *   d_out[k*p]  d_{i,j} at [i*p + j] (only filled when outer == POWER, else zeros).
 * Synchronises `cuda_stream`. */
cheb_dm_status_t cheb_dm_get_coeffs(cheb_dm_plan_t plan, double* c_out, double* g_out, double* d_out,
                                    void* cuda_stream);

/* The options the plan resolved (every "auto" replaced by the choice made: k, p, tile, fuse_sums, giant).
 * opts_out: host pointer. */
cheb_dm_status_t cheb_dm_get_options(cheb_dm_plan_t plan, cheb_dm_options_t* opts_out);

/* The block sizes chosen by the plan. */
cheb_dm_status_t cheb_dm_get_kp(cheb_dm_plan_t plan, int* k_out, int* p_out);

/* Copy the baby-step matrix T_n(X), 1 <= n <= k, of the last compute into dOut (device pointer,
 * N*N, ld N).  Test/diagnostic access to the block of Eq. (22)-(23).  Synchronises the stream. */
cheb_dm_status_t cheb_dm_get_T(cheb_dm_plan_t plan, int n, double* dOut, void* cuda_stream);

/* Chebyshev moments tau_n = tr T_n(X), n < k*p, of H (north_star item 4; reading A10):
 * bounds + rescale, baby steps, the giant block U_j = T_{jk} = T_j(T_k) (p-2 further products, kept in the
 * workspace) and tau_{jk+i} = 2 <T_{jk}, T_i>_F - tau_{jk-i} (from Eq. 7 and symmetry); all Frobenius inner
 * products are one skinny GEMM over the matrix elements on the tensor cores (gram_kernel: every matrix of
 * the two blocks is read once).  Results stay on the device inside the plan for cheb_dm_solve_mu() /
 * cheb_dm_assemble(); if tau_host != NULL (host pointer, k*p doubles) they are also copied out (this
 * synchronises the stream).  Uses the bounds mode of the last cheb_dm_coeffs() call (explicit or
 * Gershgorin); ESTATE if there was none; EUNSUPPORTED if the plan was made with moments = off. */
cheb_dm_status_t cheb_dm_moments(cheb_dm_plan_t plan, const double* dH, double* tau_host, void* cuda_stream);

/* Chemical potential for a target electron count: solves N_e(mu) = sum_n c_n(mu) tau_n = n_occ by
 * bisection on [a,b] with exactly `iters` halvings (if N_e(mid) < n_occ then lo = mid else
 * hi = mid; result (lo+hi)/2), all on the device; mu_out: host pointer.  Synchronises the stream.
 * (The kernel stops once a pass leaves [lo, hi] unchanged -- the interval has reached the spacing of the doubles and the
 * remaining halvings are no-ops -- so the result is bitwise that of `iters` halvings.)
 * ESTATE unless cheb_dm_moments() ran on this plan. */
cheb_dm_status_t cheb_dm_solve_mu(cheb_dm_plan_t plan, double beta, double n_occ, int iters,
                                  double* mu_out, void* cuda_stream);

/* mu-inclusive solve ("mu solved on the trace" of BASELINE.json's configs; adjacent to Eq. 6,
 * PAPER.md:105): bounds + rescale and the baby block T_1..T_k ONCE, the giant block U_j = T_{jk} (p-2 products),
 * moments by the Gram kernel, mu by `iters` bisection halvings on the device (N_e(mu) = n_occ, reading A9), the
 * coefficient tables for that mu (mu never leaves the device), the low-order sums G_l of Eq. (21), and
 *     D = G_0 + sum_{l=1}^{p-1} G_l U_l        (since sum_n c_n T_n = sum_l G_l T_l(T_k), reading A6)
 * as ONE long-K product (K = (p-1) N) without the serial Horner chain of Eq. (4).  k + 2p - 4 products instead
 * of the k + p - 2 of a fixed-mu solve, and nothing is computed twice.  beta and the bounds mode come from
 * cheb_dm_coeffs (its mu is ignored).  mu_out: HOST pointer (nbatch doubles for the batch form) or NULL; when
 * given, the stream is synchronised to return mu.  n_occ: target electron count(s) (HOST array for the batch
 * form).  EUNSUPPORTED if the plan was made with moments = off.
 * cheb_dm_assemble: D for NEW chemical potentials from the blocks left in the workspace by the last
 * cheb_dm_moments / cheb_dm_solve[_batch] call on the same matrices (each new mu costs the coefficient tables,
 * the sums and one long-K product -- the use in a self-consistency or MD loop); mu: HOST array of nbatch values.
 * ESTATE if no such call preceded, nbatch differs, or cheb_dm_coeffs changed the bounds (or the bounds mode) since: the
 * blocks are polynomials of X(a, b).  A new beta alone keeps them (beta is read at the call). */
cheb_dm_status_t cheb_dm_solve(cheb_dm_plan_t plan, const double* dH, double n_occ, int iters, double* dD,
                               double* mu_out, void* cuda_stream);
cheb_dm_status_t cheb_dm_solve_batch(cheb_dm_plan_t plan, int nbatch, const double* const* dH, const double* n_occ,
                                     int iters, double* const* dD, double* mu_out, void* cuda_stream);
cheb_dm_status_t cheb_dm_assemble(cheb_dm_plan_t plan, int nbatch, const double* mu, double* const* dD, void* cuda_stream);

/* One product of the recurrence as a stand-alone call (kernel-level tests and GEMM benchmark):
 *   Out = alpha * A B + beta * C,   A, B, C, Out symmetric-operand N x N device matrices (ld N),
 * computed by the same DMMA kernel as the solve (A is read through its transpose, which equals A
 * for the symmetric operands of this method).  C may be NULL (beta ignored).  Out may alias C. */
cheb_dm_status_t cheb_dm_product(cheb_dm_plan_t plan, double alpha, const double* dA, const double* dB,
                                 double beta, const double* dC, double* dOut, void* cuda_stream);

/* The same product on the Blackwell tensor path proper: sm_100a has no FP64 tcgen05 MMA, so the
 * FP64 operands are sliced error-free into S int8 digits per element (row-wise power-of-two scales), the S (S+1)/2
 * leading digit products run on tcgen05.mma kind::i8 with int32 accumulators in tensor memory, and the result is
 * recombined in FP64:  Out = alpha * A B + beta * C  with  |error_ij| <= K (S+1) 2^{-7S} max_k|a_ik| max_k|b_kj| 4
 * plus FP64 rounding of the recombination; S = 8 (36 int8 products) is below the rounding error of an FP64 dot
 * product.  A, B symmetric N x N device matrices (ld N; B may equal A), C nullable (ld N), Out must not alias A or B.
 * symmetric != 0: the caller asserts that the result is symmetric (A and B commute, C symmetric -- every product of the
 * method, whose operands are polynomials of X): only the 128 x 64 tiles that touch the lower triangle are computed and
 * each is mirrored on store.
 * Stand-alone call (kernel-level tests and benchmark against the DMMA product); with the option sliced_solve every
 * product of the solve runs through the same two kernels.
 * EUNSUPPORTED unless the plan was made with the option sliced = S. */
cheb_dm_status_t cheb_dm_product_sliced(cheb_dm_plan_t plan, double alpha, const double* dA, const double* dB,
                                        double beta, const double* dC, double* dOut, int symmetric, void* cuda_stream);

/* Synchronises `cuda_stream` and reports what the device flagged since the last check (the flags are sticky, so one
 * check after a pipeline of computes sees an error of any of them; the check clears them): CHEB_DM_ECUDA if a CUDA
 * error is pending or a dependency wait inside a persistent kernel hit its watchdog (~4 s; never in a correct
 * run), CHEB_DM_EBOUNDS for non-finite bounds, CHEB_DM_ENOCONV for the stability guard of the power-basis outer
 * recursion, else CHEB_DM_OK.  cheb_dm_compute_host() and cheb_dm_wait() perform the same check. */
cheb_dm_status_t cheb_dm_check(cheb_dm_plan_t plan, void* cuda_stream);

/* Bytes of device workspace owned by the plan. */
cheb_dm_status_t cheb_dm_workspace_bytes(cheb_dm_plan_t plan, size_t* bytes_out);

/* Number of kernel launches issued by the last cheb_dm_compute[_batch] / cheb_dm_solve[_batch] / cheb_dm_assemble /
 * cheb_dm_moments call (for bench.py's gpu_launches). */
cheb_dm_status_t cheb_dm_last_launch_count(cheb_dm_plan_t plan, int* launches_out);

/* Executed FP64 tensor flops of one cheb_dm_compute() of ONE matrix on this plan: 2*N^3 per product, only the
 * computed tiles with symmetric-tile skipping.  cheb_dm_flops_per_solve: the same for cheb_dm_solve (baby block,
 * giant block, Gram kernel and the long-K assembly). */
cheb_dm_status_t cheb_dm_flops_per_compute(cheb_dm_plan_t plan, double* flops_out);
cheb_dm_status_t cheb_dm_flops_per_solve(cheb_dm_plan_t plan, double* flops_out);
/* Executed int8 tensor operations of one cheb_dm_compute() on a plan with sliced_solve: products x S (S+1)/2 digit
 * products x 2 x (computed 128 x 64 tiles) x kpad.  EUNSUPPORTED without the option. */
cheb_dm_status_t cheb_dm_sliced_ops_per_compute(cheb_dm_plan_t plan, double* ops_out);

/* Measurement support (bench.py's roofline object).
 * cheb_dm_set_timing(plan, 1): every following cheb_dm_compute() records a CUDA event on its stream
 *   directly before and after the launches of the product kernels (GROUPED mode: one persistent launch, or
 *   baby-step launch + [form_sums_kernel] + giant-step launch).
 *   The plan keeps a ring of 256 event pairs, so up to 256 computes can be in flight unsynchronised.
 * cheb_dm_product_ms: waits for the recorded computes (the last min(count, 256) since timing was
 *   switched on) and returns how many there were and the SUM of their product-launch durations in
 *   milliseconds (host pointers).  ESTATE if timing is off or nothing ran.
 * cheb_dm_dmma_peak: register-resident DMMA.8x8x4 issue-rate microbenchmark on all SMs (the FP64
 *   tensor roofline of this device at its current clocks): `iters` dependent steps of 8 independent
 *   accumulator chains per warp, 32 warps per SM; tflops_out: host pointer.  Synchronises the stream. */
cheb_dm_status_t cheb_dm_set_timing(cheb_dm_plan_t plan, int enable);
cheb_dm_status_t cheb_dm_product_ms(cheb_dm_plan_t plan, int* count_out, double* total_ms_out);
cheb_dm_status_t cheb_dm_dmma_peak(int iters, double* tflops_out, void* cuda_stream);

/* Per-tile timeline of the persistent product kernel (tracing aid).
 * cheb_dm_set_trace(plan, 1): following launches record, per work item (one output tile of one product), the
 *   %globaltimer nanoseconds at which the producer claimed it, the consumer warps received it, its first operand
 *   stage landed, its K loop ended and its result was published, plus the SM it ran on.  Costs a few
 *   instructions per tile; EALLOC if the record buffer cannot be allocated.
 * cheb_dm_get_trace: copies the records of the last cheb_dm_compute() (items in claim order: baby-step tasks
 *   first, then giant steps; at most max_records) to HOST memory `out`, count to *count_out (host).
 *   Synchronises the device.  ESTATE if tracing was never enabled. */
typedef struct {
    int task, tm, tn, sm;
    unsigned long long t_claim, t_desc, t_first, t_kend, t_done;
} cheb_dm_trace_rec_t;
cheb_dm_status_t cheb_dm_set_trace(cheb_dm_plan_t plan, int enable);
cheb_dm_status_t cheb_dm_get_trace(cheb_dm_plan_t plan, cheb_dm_trace_rec_t* out, int max_records, int* count_out);

/* Step a-1 for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the Gershgorin bounds of PAPER.md:96 (readings A1, A2-iv) WITHOUT a plan and without any
 * allocation.  It is a variant of the bounds pass of the front-end kernel whose scratch (one (h_ii - R_i, h_ii + R_i)
 * pair per row, R_i = sum_{j != i} |h_ij|, and a completion ticket) lives in a file-scope static device array of
 * 256 + 16 * CHEB_DM_STATIC_MAX_N bytes (129 KiB) that every GPU that loads the library holds until exit.
 *   dH       DEVICE, symmetric N x N, leading dimension ldh >= N (elements); read only.
 *   d_bounds DEVICE, 2 doubles: (a, b) = (min_i (h_ii - R_i), max_i (h_ii + R_i)); a == b is widened to (a - 1, b + 1) as
 *            in the solve; a non-finite row gives (-inf, +inf).
 * One kernel launch on `cuda_stream` (plus a 256-byte cudaMemsetAsync of the ticket, which must start at zero); no
 * synchronisation; calls no cudaMalloc, cudaFree or allocating library routine (the array's device address is looked
 * up with cudaGetSymbolAddress once per device, at the first call on that device).
 * N > CHEB_DM_STATIC_MAX_N -> CHEB_DM_ESIZE (nothing launched); N < 1, NULL pointers, ldh < N -> CHEB_DM_EINVAL.
 * ALL calls on a device share the one array, which keeps the last call's contents: calls that overlap on the GPU
 * (different streams, or graph branches) race -- serialise them. */
#define CHEB_DM_STATIC_MAX_N 8192
cheb_dm_status_t cheb_dm_bounds_static(const double* dH, int N, long long ldh, double* d_bounds, void* cuda_stream);

const char* cheb_dm_strerror(cheb_dm_status_t status);

#ifdef __cplusplus
}
#endif
#endif /* CHEB_DM_H */
