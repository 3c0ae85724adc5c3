/* hsp.h -- C-ABI boundary of the B200-native Horseshoe-Probit Gibbs sweep.
 *
 * Method: Terenin, Dong & Draper, "GPU-accelerated Gibbs sampling: a case study of the Horseshoe
 * Probit model" (arXiv 1608.04329).  Citations are PAPER.md:<line> (+ section / equation).
 *
 * Problem statement the calls follow: inputs are the N x p design matrix X ("the (n x p) matrix
 * whose rows are the vectors x_i") and y in {0,1}^N; a chain is run
 * from the cold start beta=0, lambda=nu=tau=xi=1 for n iterations of the sweep
 * of PAPER.md:188-189 with the full conditionals of eq. (12); the outputs are
 * the Monte Carlo draws of beta, lambda, tau.
 *
 * One sweep (k <- k+1), every step a CUDA kernel of this library (no CPU fallback exists):
 *   a1  eta_i = x_i . beta
 *   a2  z_i ~ TN(eta_i, 1) on the side of 0 fixed by y_i
 *   a3  per-CTA partials of X^T z from the same on-chip tile PAPER.md:200
 *   b   g = deterministic fixed-order sum of the partials
 *   e1  lam_j^-2 = -ln u / (nu_j^-1 + tau^-2 beta_j^2 / 2)   PAPER.md:176, 224   (old beta, tau^-2)
 *   e2  tau^-2 = Gamma((p+1)/2) / (xi^-1 + 1/2 sum lam_j^-2 beta_j^2), Cheng (1977)
 *   c   Q = X^T X + diag(tau^-2 lam_j^-2)                    PAPER.md:186, 196  (X^T X once, at create)
 *   d1  Q = L L^T  (blocked fp64 Cholesky)
 *   d2  beta = Q^-1 g + L^-T e,  e ~ N(0, I)
 *   e3  nu_j^-1 = -ln u / (1 + lam_j^-2);  xi^-1 = -ln u / (1 + tau^-2)
 *   g   append beta, lambda_j = (lam_j^-2)^-1/2, tau = (tau^-2)^-1/2 to the device history
 * Random numbers: Philox-4x32-10, counter (idx_lo, idx_hi, sweep k, tag), key =
 * seed; one call per variate, so results do not depend on grid shape (DESIGN.md "Random-number
 * contract").  State, sampler, Gram, Q and L are fp64 whatever the dtype of X.
 *
 * Conventions: every call returns an int status (HSP_OK = 0, negative = error), never throws and
 * never aborts; hsp_last_error() gives a thread-local message for the last failing call.  All
 * device work is enqueued on the stream given at create; calls that copy results out synchronise
 * that stream.  "DEVICE" / "HOST" below says where a pointer must live; "ANY" means host or device
 * (cudaMemcpyDefault).
 */
#ifndef HSP_H_
#define HSP_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hsp_state hsp_state; /* opaque; owned by the library; free with hsp_destroy */

enum { HSP_F32 = 0, HSP_F64 = 1 };
enum { HSP_OK = 0, HSP_EINVAL = -1, HSP_ENOMEM = -2, HSP_ECUDA = -3, HSP_ENOTPD = -4, HSP_ENUMERIC = -5 };
/* flags for hsp_set_flags (default: 0) */
enum {
  HSP_STORE_Z = 1u,       /* a2 also writes z (fp64, N) to a device buffer for hsp_get_latent      */
  HSP_FREEZE_SCALES = 2u, /* skip e1, e2, e3 (lambda, tau, nu, xi keep their current values)       */
  HSP_FREEZE_Z = 4u,      /* skip a1-a3 and b (g keeps the value of the last sweep that ran them)   */
  HSP_FREEZE_BETA = 16u,  /* skip c, d1, d2 (beta keeps its current value)                          */
  HSP_NO_GRAPH = 32u,     /* enqueue kernels directly instead of replaying the captured CUDA graph  */
  HSP_SERIAL = 64u,       /* one stream: no overlap of the Cholesky branch with the fused pass      */
  HSP_PAPER_DESIGN = 128u /* A/B: rows a1-a3 by the paper's own decomposition: X beta, a
                             divergent rejection sampler (thread per row), X^T z -- X is read twice, mu and z go
                             through HBM; same law as the fused pass, different draws (implies HSP_STORE_Z)       */
};

/* Create a chain.  PAPER.md:186 (X, y), PAPER.md:289 (cold start), PAPER.md:195 (X^T X once).
 *   out     HOST   receives the handle (NULL on error).
 *   X       DEVICE row-major N x p, dtype x_dtype (HSP_F32 | HSP_F64), 16-byte aligned, row pitch
 *                  p * sizeof(elem).  BORROWED: never copied, never written; the caller keeps it
 *                  alive until hsp_destroy.
 *   y       DEVICE N bytes, each 0 or 1.  BORROWED likewise.  Any other value -> HSP_EINVAL.
 *   N >= 2, p >= 1, seed any 64-bit value.
 *   stream  cudaStream_t passed as void* (NULL = the legacy default stream).
 * Computes G = X^T X (fp64 result) on the stream and returns after it has completed: fp64 X and small problems by
 * exact fp64 products; fp32 X with N p^2 >= 2e10 on the tcgen05 tensor cores (split-bf16 products, fp64 flush:
 * |dG| <= 1e-6 max|G|; option "gram_tc" forces either).  The launch plan (kernel variant, tile shape, SMs of the
 * Cholesky branch) is fixed here from (N, p, dtype) and the plan-time options in force (hsp_set_option).
 * One process may hold chains on several devices: the chain lives on the device current at create.
 * Errors: HSP_EINVAL (arguments), HSP_ENOMEM, HSP_ECUDA.                                        */
int hsp_create(hsp_state** out, const void* X, int x_dtype, const unsigned char* y, long long N, int p,
               unsigned long long seed, void* stream);

/* Same, but X and y are HOST buffers (pinned or pageable): the library allocates device copies it
 * owns, uploads them on the stream (this is the end-to-end entry bench.py times) and frees them in
 * hsp_destroy.                                                                                   */
int hsp_create_host(hsp_state** out, const void* X_host, int x_dtype, const unsigned char* y_host,
                    long long N, int p, unsigned long long seed, void* stream);

/* Row-sharded chains (the z_i are conditionally independent, so the rows of
 * X split across GPUs).  Each rank creates a chain on ITS rows; row_offset = global index of its first row, so
 * that the Philox counter of z_i is the global row and the draws do not depend on the number of ranks.  After
 * create, the caller sums hsp_gram_device (p*p doubles) over the ranks, in place, once.  Then, per sweep:
 *   hsp_sweep_begin   enqueues a1-a3, b on the local rows (-> hsp_xtz_device, p doubles) and e1-e3, c, d1
 *   <caller>          sums hsp_xtz_device over the ranks in place (one all-reduce of p doubles, e.g. NCCL on the
 *                     same stream); every rank then holds the same X^T z bit for bit
 *   hsp_sweep_end     enqueues d2: every rank draws the same beta (same counters, same inputs)
 * hsp_sweep_prepare(n) reserves the history for the next n begin/end pairs (what hsp_get_draws returns).
 * All asynchronous on the stream; no host synchronisation per sweep.  X, y DEVICE, borrowed, as in hsp_create.
 * Errors as hsp_create / hsp_sweep; HSP_EINVAL if the calls are made out of order.                  */
int hsp_create_shard(hsp_state** out, const void* X, int x_dtype, const unsigned char* y, long long N_local,
                     int p, unsigned long long seed, long long row_offset, void* stream);
int hsp_sweep_prepare(hsp_state* s, long long n_iter);
int hsp_sweep_begin(hsp_state* s);
int hsp_sweep_end(hsp_state* s);
double* hsp_xtz_device(hsp_state* s);   /* DEVICE, p doubles, owned by the library   */
double* hsp_gram_device(hsp_state* s);  /* DEVICE, p*p doubles row-major (symmetric) */

/* Run n_iter sweeps (steps a1..g above, in the order PAPER.md:188-189 fixes), asynchronously on the
 * stream.  The draws of this call replace the history of the previous call.  n_iter >= 0.
 * Errors: HSP_EINVAL, HSP_ENOMEM (history n_iter*(2p+1)*8 bytes), HSP_ECUDA.  A Cholesky breakdown
 * or non-finite state inside the sweeps is reported by the next synchronising call
 * (hsp_get_draws / hsp_get_state / hsp_sync) as HSP_ENOTPD / HSP_ENUMERIC.                       */
int hsp_sweep(hsp_state* s, long long n_iter);
/* Reserve device history for calls of up to n_iter sweeps (it only grows).  hsp_sweep grows it on demand, which
 * synchronises the chain and allocates: a caller that times its sweeps, or must not allocate later, reserves first.
 * The draws of the previous hsp_sweep call are discarded when the history grows.  Errors: HSP_EINVAL, HSP_ENOMEM.   */
int hsp_reserve_history(hsp_state* s, long long n_iter);

/* Copy the draws of the most recent hsp_sweep call: beta[n_iter*p],
 * lambda[n_iter*p], tau[n_iter], row-major by sweep.  ANY pointers; any may be NULL.
 * Synchronises the stream.                                                                       */
int hsp_get_draws(const hsp_state* s, double* beta, double* lambda, double* tau);

/* Asynchronous download of the Monte Carlo output ("Monte Carlo output is downloaded off of the GPU
 * at the same time as updates for other variables are computed").  Registers a HOST ring of `capacity` sweeps:
 * host_beta[capacity*p], host_lambda[capacity*p], host_tau[capacity] (any may be NULL; BORROWED until the next
 * hsp_set_output / hsp_destroy; pinned memory -- cudaHostAlloc / cudaHostRegister -- keeps the copies asynchronous).
 * From then on every sweep enqueued by hsp_sweep / hsp_sweep_end is also copied to ring row (r mod capacity), r = 0,
 * 1, ... counting sweeps since this call, by a copy stream that waits on an event recorded after the sweep's beta
 * draw -- in blocks of a few sweeps (>= 64 KB), with no host synchronisation and without delaying the next sweep.
 * capacity = 0 or all pointers NULL switches the download off.  hsp_get_draws is unaffected.
 *   hsp_output_ready  non-blocking: *rows = number of sweeps (since hsp_set_output) that have landed on the host.
 *   hsp_output_wait   blocks until every sweep enqueued so far has landed; *rows (may be NULL) = their number;
 *                     returns the device status like hsp_sync (HSP_ENOTPD / HSP_ENUMERIC).
 * Errors: HSP_EINVAL, HSP_ECUDA.                                                                  */
int hsp_set_output(hsp_state* s, double* host_beta, double* host_lambda, double* host_tau, long long capacity);
int hsp_output_ready(hsp_state* s, long long* rows);
int hsp_output_wait(hsp_state* s, long long* rows);

/* Synchronise the stream and report device-side status (HSP_OK, HSP_ENOTPD, HSP_ENUMERIC).       */
int hsp_sync(const hsp_state* s);

int hsp_destroy(hsp_state* s);

/* Thread-local message of the last call that failed on this thread ("" if none).                 */
const char* hsp_last_error(void);

/* ---- debug / test / measurement entry points ------------------------------------------------ */

/* z of the last sweep (needs HSP_STORE_Z set before that sweep, else HSP_EINVAL) and the truncation
 * side 2y-1.  ANY pointers, may be NULL.  Synchronises.                           */
int hsp_get_latent(const hsp_state* s, double* z, signed char* side);
/* Current state; p-vectors and scalars, ANY pointers, may be NULL.  sweep = number of sweeps done. */
int hsp_get_state(const hsp_state* s, double* beta, double* lam_inv2, double* nu_inv, double* tau_inv2,
                  double* xi_inv, long long* sweep);
/* Overwrite parts of the state (NULL = keep; sweep < 0 = keep).  Because the random numbers are a
 * pure function of (seed, index, sweep, tag), get_state/set_state give exact checkpoint/resume.   */
int hsp_set_state(hsp_state* s, const double* beta, const double* lam_inv2, const double* nu_inv,
                  const double* tau_inv2, const double* xi_inv, long long sweep);
int hsp_set_flags(hsp_state* s, unsigned flags);
/* g = X^T z of the last sweep (p), G = X^T X (p*p, row-major, lower triangle valid), L (p*p, lower). */
int hsp_get_xtz(const hsp_state* s, double* g);
int hsp_get_gram(const hsp_state* s, double* G);
int hsp_get_chol(const hsp_state* s, double* L);
/* Average device time (ms) of the fused pass a1-a3 over the launches since the last call of this
 * function, measured with CUDA events on the launching stream when HSP_NO_GRAPH is set; and the
 * number of launches averaged.  Synchronises.                                                    */
int hsp_get_fused_pass_ms(hsp_state* s, double* ms, long long* launches);
/* Number of kernels this library launched (directly or through graph replays) since create.      */
long long hsp_get_launch_count(const hsp_state* s);
/* Launch plan chosen at create: CTAs of the fused pass (a1-a3), CTAs of the Cholesky branch (c, d1),
 * whether the two run side by side on disjoint SMs (1) or one after the other (0), and the cost-model
 * estimate of the Cholesky branch in microseconds.  HOST pointers, any may be NULL.               */
int hsp_get_plan(const hsp_state* s, int* fused_ctas, int* chol_ctas, int* overlap, double* chol_est_us);
/* Name of the fused-pass kernel variant selected for this (dtype, N, p): "tma" (rows of >= 128 16-byte vectors),
 * "tma-narrow" (narrower rows, p <= 511, X >= 2 MB) or "generic" (everything else).                */
const char* hsp_fused_variant(const hsp_state* s);

/* Plan-time and launch-mode options (tests and tuning; the defaults are what bench.py measures).  The library reads
 * NO environment variables.  state == NULL sets the process-wide default that chains created AFTERWARDS copy at
 * create (thread-safe); value < 0 restores the automatic choice; key == NULL (state == NULL) restores all.  With a
 * state only "no_pdl" may change (the launch plan of an existing chain is fixed).  Keys:
 *   fused_eta 0|2      eta arithmetic for fp32 X: exact fp64 | fp32 chains of 4 (default)
 *   fused_grid, fused_stages, fused_lag, fused_w (256|512), narrow_rt      grid, ring depth, lag, threads across a
 *                      row, rows per narrow tile of the fused pass
 *   fused_variant 0|1  force the generic kernel | allow the wide TMA kernel below 128 vectors per row
 *   fused_narrow 0     disable the narrow kernel
 *   chol_ctas K, chol_sb (tiles per inverse super-block), chol_trace 1     Cholesky branch
 *   gram_tc 0|1        exact | tensor-core Gram
 *   no_pdl 1           tail kernels without programmatic dependent launch
 * Errors: HSP_EINVAL (unknown key, plan-time key with a state).                                     */
int hsp_set_option(hsp_state* s, const char* key, long long value);
int hsp_get_option(const hsp_state* s, const char* key, long long* value);

/* Rows a1-a3 + b as ONE stateless call that ALLOCATES NOTHING (no cudaMalloc / cudaFree, no allocating library routine), for
 * callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid it.  For a given
 * beta and sweep number k it computes eta = X beta, z_i ~ TN(eta_i, 1) on the side fixed by y_i with the Philox
 * counters (i, k, Z) of the chain, and g = X^T z -- the same kernels as hsp_sweep, the same
 * values as a chain with that seed whose state is beta at sweep k.
 *   X, y    DEVICE, as for hsp_create (y is NOT validated here: every byte must be 0 or 1)
 *   beta    DEVICE p doubles (read);  g_out  DEVICE p doubles (written);  z_out  DEVICE N doubles or NULL
 *   k       sweep number, 1 <= k < 2^32;  stream: cudaStream_t as void* (NULL = the legacy default stream)
 * Scratch (per-CTA partials of X^T z, control block) lives in a static device array of hsp_noalloc_scratch_bytes() = 8 MiB +
 * 256 B that every GPU which loads the library holds until the process exits.  Limit: (CTAs x row groups of the pass) x p <=
 * 2^20 doubles -- on 148 SMs: p <= 7084 with the wide TMA kernel, any p <= 511 with the narrow one, p <= 1771 with the generic
 * kernel (wide rows that are not a multiple of 16 bytes); larger problems get
 * HSP_EINVAL (message: hsp_noalloc_last_error) and must use hsp_create / hsp_sweep.  All calls share the array: calls that
 * overlap on the GPU (two streams, two host threads) RACE -- serialise them.  Asynchronous: returns after enqueueing.
 * Errors: HSP_EINVAL, HSP_ECUDA.                                                                                       */
int hsp_xtz_noalloc(const void* X, int x_dtype, const unsigned char* y, long long N, int p, unsigned long long seed,
                    long long k, const double* beta, double* g_out, double* z_out, void* stream);
long long hsp_noalloc_scratch_bytes(void);
const char* hsp_noalloc_last_error(void);

/* Device unit-test hooks (one thread per element; DEVICE pointers):
 *   philox : out[4n] = Philox-4x32-10(ctr[4n], key[2n])
 *   uniform: ua[n], ub[n] from (seed, idx[n], sweep, tag) -- the variate addressing of the sweep
 *   tnpos  : w[n] = TNpos(m[n], u[n]);   norm_inv: x[n] = Phi^-1(u[n])
 *   cheng  : x[n] = Gamma(alpha, 1) drawn with (seed, sweep = sweep0 + i)                         */
int hsp_dbg_philox(const unsigned* ctr, const unsigned* key, unsigned* out, long long n, void* stream);
int hsp_dbg_uniform(unsigned long long seed, const unsigned long long* idx, unsigned sweep, unsigned tag,
                    double* ua, double* ub, long long n, void* stream);
int hsp_dbg_tnpos(const double* m, const double* u, double* w, long long n, void* stream);
int hsp_dbg_norm_inv(const double* u, double* x, long long n, void* stream);
int hsp_dbg_cheng(double alpha, unsigned long long seed, unsigned sweep0, double* x, long long n, void* stream);


/* Measurement hook for rows c, d1: the static schedule of the Cholesky task graph and, if
 * option "chol_trace" = 1 was in force when the chain was created, the device timestamps of
 * the tasks of the last sweep.  rows: HOST, capacity x 12 long long per task, in schedule order:
 * {type, i, j, kbeg, kend, slot_in, slot_out, cta, t_start_ns, t_kloop_end_ns, t_end_ns, 0} (timestamps 0
 * without the trace; chain task POTRF, type 2: t_kloop_end_ns = end of the tile factorisation and the last word = end of
 * the triangular inverse).  Returns the number of tasks (rows may be NULL to query it), or a negative status.
 * Synchronises.                                                                                     */
long long hsp_dbg_chol_trace(const hsp_state* s, long long* rows, long long capacity);
/* Host-only (no device needed): the static schedule the library would build for nt tile rows (64 x 64 tiles), inverse
 * super-blocks of sb tiles and K CTAs.  rows: HOST, capacity x 8 int per task, the K per-CTA lists concatenated:
 * {cta, type, i, j, kbeg, kend, slot_in, slot_out}; task types: 0 tile L(i,j) (prefix when slot_out >= 0), 1 inverse
 * tile W(j,i), 2 / 3 / 4 the chain tasks POTRF(j), TRSM(j) -> L(j+1,j), SYRK(j) -> A(j+1,j+1) of the first list.
 * makespan_us (may be NULL): the cost-model estimate.  Returns the number of tasks (rows may be NULL to query
 * it) or HSP_EINVAL.                                                                                */
long long hsp_dbg_chol_schedule(int nt, int sb, int K, int* rows, long long capacity, double* makespan_us);

#ifdef __cplusplus
}
#endif
#endif /* HSP_H_ */
