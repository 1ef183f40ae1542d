/*
 * alora.h -- C ABI of libalora: the data-parallel hot path of ALORA (arXiv 2505.15775), the
 * rank-adaptive augmented-Lagrangian / Burer-Monteiro solver for low-rank SDPs, as sm_100a CUDA.
 *
 * Problem (P), PAPER.md:85-91 (sec. 1.2):   min <C,X>  s.t.  [A(X)]_i = <A_i,X> = b_i (i<m),  X psd.
 * ALM-BM subproblem (AL-BM), with X = R R^T, R in R^{n x r}
 * (the paper's F, rho, L-bar are R, sigma, f here):
 *     f(R)    = <C,RR^T> - y^T q + (sigma/2)||q||^2,        q = A(RR^T) - b
 *     grad f  = 2 S(lambda) R,   S(w) = C - A^*(w) = C - sum_i w_i A_i,   lambda = y - sigma q
 *               ("nabla h(F) = 2 nabla f(X) F"; :483 z_{y,rho}; :111 Z(y))
 *
 * Storage convention for all sparse symmetric matrices: SYM-UPPER COO -- an entry (j,k,a) with
 * j <= k means A[j,k] = A[k,j] = a; duplicates are summed; explicit zeros are kept.  "X_jk = c" is
 * therefore the single entry (j,k,1/2), as in the paper's examples.
 *
 * Conventions.  Every call returns an alora_status and never throws or aborts; on error the
 * outputs are unspecified and nothing is freed.  "HOST"/"DEVICE" says where a pointer lives.
 * Device buffers passed in (R, D, G, V, W, y, z, mu) are caller-owned; the library owns only its
 * device copy of the problem and its workspace.  All work is enqueued on the stream given at
 * create; calls that return host scalars synchronise that stream before returning, calls that do
 * not (documented per call) return as soon as the work is enqueued.  A ctx is not thread-safe.
 * Reductions are two-stage and ordered, so results are bit-reproducible run to run.
 * There is no CPU fallback: without a CUDA device alora_create fails with ALORA_ECUDA.
 */
#ifndef ALORA_H
#define ALORA_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct alora_ctx alora_ctx; /* opaque: one per (problem, dtype, device, stream) */

typedef enum {
  ALORA_OK = 0,
  ALORA_EINVAL = 1,  /* bad argument (index out of range, row > col, non-monotone A_ptr, NaN, r too large, misaligned) */
  ALORA_ENOMEM = 2,  /* host or device allocation failed */
  ALORA_ECUDA = 3,   /* CUDA runtime error (text in alora_last_error) */
  ALORA_ESTATE = 4,  /* call order violated (e.g. alora_eval before alora_set_dual) */
  ALORA_ENOTCONV = 5 /* alora_solve / alora_lanczos hit its iteration cap; outputs are the last iterate */
} alora_status;

/* dtype of R/D/G/V/W and of the library's copy of the stored values.  Products are formed in this
 * type; every sum over rows / constraints and y, b, z, lambda, mu are always fp64. */
typedef enum { ALORA_F32 = 0, ALORA_F64 = 1 } alora_dtype;

typedef struct {
  int64_t n, m;
  /* cost C: sym-upper COO */
  int64_t nnzC;
  const int32_t *C_row, *C_col;
  const double *C_val;
  /* optional low-rank cost term  C += U diag(s) U^T;  U is n x pC COLUMN-major, pC <= 8; NULL if pC == 0 */
  int32_t pC;
  const double *C_U, *C_s;
  /* constraints: stacked sym-upper COO, entries [A_ptr[i], A_ptr[i+1]) belong to A_i */
  int64_t nnzA;
  const int64_t *A_ptr; /* m+1, monotone, A_ptr[0] = 0, A_ptr[m] = nnzA */
  const int32_t *A_row, *A_col;
  const double *A_val;
  const double *b; /* m */
} alora_problem;   /* all HOST pointers, caller-owned, copied (and re-laid-out) at create */

/* Validates (0 <= row <= col < n, monotone A_ptr, finite values -> ALORA_EINVAL), copies the problem
 * to `device` and builds the row-oriented layouts.  `cuda_stream` is a cudaStream_t (NULL = default
 * stream).  On failure *out is NULL and alora_strerror(status) describes the class of error. */
alora_status alora_create(const alora_problem *p, alora_dtype dtype, int device, void *cuda_stream,
                          alora_ctx **out);
void alora_destroy(alora_ctx *ctx); /* NULL is allowed */
const char *alora_last_error(const alora_ctx *ctx); /* detail of the last failure; valid until the next call on ctx */
const char *alora_strerror(alora_status s);

/* info[0]=class (0: "diagonal" class -- every A_i is one diagonal entry and no row carries two, e.g.
 * MaxCut: f and grad run as ONE fused pass; 1: general class -- forward pass, then adjoint pass),
 * [1]=n, [2]=m, [3]=stored off-diagonal entries of C (full pattern), [4]=entries of the row-oriented
 * constraint pattern (full), [5]=entries of the forward (sym-upper) constraint list, [6]=number of
 * "long" constraints (split across blocks), [7]=kernel launches issued by this ctx so far,
 * [8]=device bytes held by the ctx, [9]=number of SMs. */
alora_status alora_info(const alora_ctx *ctx, int64_t info[16]);

/* Dual vector y (DEVICE fp64[m], caller-owned, read by every later call until replaced) and penalty
 * sigma > 0 (paper: rho).  Does not synchronise. */
alora_status alora_set_dual(alora_ctx *ctx, const double *y_dev, double sigma);

/* f(R) and G = grad f(R).
 * R, G: DEVICE, dtype of the ctx, row-major n x r with leading dimension ld >= r (elements).
 *   Vector width follows alignment: 16-byte loads when the base pointers and ld*sizeof(elem) are
 *   multiples of 16, else 8, else element-wise.  r <= 64 always works; up to 256 (f32) / 128 (f64)
 *   with 16-byte alignment.  G must not alias R.  G may be NULL (value-only call).
 * z_dev: DEVICE fp64[m] receiving z = A(RR^T), or NULL (then kept in the ctx).
 * stats: HOST double[8] or NULL.  [0]=f, [1]=<C,RR^T>, [2]=y.q, [3]=||q||^2, [4]=||G||_F^2,
 *   [5]=<G,R>, [6]=lambda.z, [7]=0.  If stats != NULL the call synchronises the stream; if NULL it
 *   only enqueues (fetch later with alora_get_stats). */
alora_status alora_eval(alora_ctx *ctx, const void *R, int32_t r, int64_t ld, void *G, double *z_dev,
                        double stats[8]);
alora_status alora_get_stats(alora_ctx *ctx, double stats[8]); /* of the last alora_eval; synchronises */

/* lambda = y - sigma (z - b) of the last alora_eval into lam_dev (DEVICE fp64[m]).
 * Enqueues only. */
alora_status alora_get_lambda(alora_ctx *ctx, double *lam_dev);

/* Helpers for callers that assemble z = A(RR^T) themselves -- the row-sharded evaluation of
 * paper_2505_15775_b200/sharded.py, where z is the sum over ranks of the partial z of each rank's entries and a rank
 * owns a block of rows.
 * alora_dual_terms: q = z - b, lambda = y - sigma q with the (y, sigma) of alora_set_dual, for the
 *   caller's z_dev (DEVICE fp64[m]); lam_dev (DEVICE fp64[m]) receives lambda or is NULL; out: HOST double[3] =
 *   {y.q, ||q||^2, lambda.z}.
 * alora_rowdots: out (HOST double[2]) = {sum X_ij^2, sum X_ij Y_ij} over the first n_rows rows of X, Y (DEVICE, ctx
 *   dtype, row-major with r columns and leading dimension ld).
 * Both synchronise. */
alora_status alora_dual_terms(alora_ctx *ctx, const double *z_dev, double *lam_dev, double out[3]);
alora_status alora_rowdots(alora_ctx *ctx, const void *X, const void *Y, int64_t n_rows, int32_t r, int64_t ld,
                           double out[2]);

/* Allocation-free variant of alora_rowdots, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it): the same two sums, out_dev[0] = sum X_ij^2, out_dev[1] = sum X_ij Y_ij
 * over the first n_rows rows, but the per-block partial sums live in a static __device__ array inside the library
 * (about 64 KB, held by every GPU that loads the library until the process exits) instead of the ctx workspace, and
 * the result goes to out_dev (DEVICE double[2], caller-owned).  The call makes no cudaMalloc / cudaFree, calls no
 * allocating library routine and does not synchronise: it enqueues one 4-byte memset and one kernel on the ctx stream.
 * Limit: n_rows * r <= ALORA_ROWDOTS_STATIC_MAX_ELEMS (the array holds one partial row per 16384 elements); larger
 * shapes are rejected with ALORA_EINVAL and a message naming the limit -- use alora_rowdots for them.  The first call on
 * a device looks up the array's device address (no allocation; make that first call outside a stream capture).
 * The array is shared by every call on the device and keeps the last call's contents (the call clears what must start
 * at zero itself); calls that overlap on the GPU -- two streams, or two ctx on one device used concurrently -- race on
 * it and must be serialised by the caller.  Summation order differs from alora_rowdots (fixed 16384-element chunks,
 * independent of the SM count), so the two agree to fp64 rounding, not bit for bit. */
#define ALORA_ROWDOTS_STATIC_MAX_ELEMS 67108864 /* 2^26 */
alora_status alora_rowdots_static(alora_ctx *ctx, const void *X, const void *Y, int64_t n_rows, int32_t r, int64_t ld,
                                  double *out_dev);

/* Same as alora_eval but R, G, z are HOST buffers (G, z may be NULL): copies R to the device,
 * evaluates, copies G and z back, inside the call.  stats as above (must be non-NULL). */
alora_status alora_eval_host(alora_ctx *ctx, const void *R_host, int32_t r, int64_t ld, void *G_host,
                             double *z_host, double stats[8]);

/* One whole step of the hot path with HOST buffers (bench.py's end-to-end leg): f + grad at R, the line-search
 * coefficients along D (warm form) and W = S(lambda) V with lambda of that evaluation.  R_host, D_host (n x r, ld),
 * V_host (n): inputs; G_host (n x r, ld), z_host (fp64[m]), W_host (n): outputs, each may be NULL.  All HOST, ctx
 * dtype; page-locked memory makes the copies asynchronous.  The copies run inside the call and are overlapped with
 * the kernels where the data flow allows (D goes up while f + grad runs and G comes down; G, z come down on a
 * second stream while the line search runs).  stats[8], p[5], vw as in the device calls (non-NULL).  Synchronises. */
alora_status alora_step_host(alora_ctx *ctx, const void *R_host, const void *D_host, const void *V_host, int32_t r,
                             int64_t ld, void *G_host, double *z_host, void *W_host, double stats[8], double p[5],
                             double *vw);

/* Exact line search: coefficients p[0..4] (HOST) of alpha -> f(R + alpha D) = sum_k p_k alpha^k, from
 * q = A(RR^T)-b, q1 = A(RD^T+DR^T), q2 = A(DD^T) expanded in (AL-BM):
 *   p0 = f(R), p1 = 2<C,RD^T> - y.q1 + sigma q.q1 = <G,D>, p2 = <C,DD^T> - y.q2 + (sigma/2)|q1|^2 + sigma q.q2,
 *   p3 = sigma q1.q2, p4 = (sigma/2)|q2|^2.
 * R, D as in alora_eval.  Synchronises.  p == NULL: enqueue only; fetch with alora_get_linesearch.
 * warm == 0 ("cold", what bench.py times): correct whatever was called before -- q is recomputed from R.
 * warm != 0: the caller states that the ctx still holds the state of an alora_eval on this same R (same pointer,
 *   r, ld, same y and sigma, R not written since); the library may then reuse that state instead of recomputing
 *   it (p0 is taken from the evaluation's f, and q-only sums from its scalars).  ALORA_ESTATE if no such evaluation
 *   is on record (different R pointer / r / ld, or alora_set_dual called since).  Results equal the cold form to
 *   rounding.  If that evaluation wrote a gradient G (G != NULL there, and != D here), the caller also vouches that G
 *   has not been written since: for the diagonal class the library then streams G and takes p1 = <G,D> -- the
 *   directional derivative -- and <C,RR^T> from the evaluation, so the pass gathers only the D operand of each
 *   neighbour pair, half the random row reads of the cold form. */
alora_status alora_linesearch(alora_ctx *ctx, const void *R, const void *D, int32_t r, int64_t ld, int32_t warm,
                              double p[5]);
alora_status alora_get_linesearch(alora_ctx *ctx, double p[5]);

/* W = S(mu) V = (C - A^*(mu)) V  (the operator of Alg. 1 line 5, with
 * mu = lambda, and of eq. 77, with mu = y).  mu_dev: DEVICE fp64[m], or NULL = lambda = y - sigma q of
 * the last alora_eval (recomputed from that evaluation's z -- if the caller passed its own z_dev there,
 * that buffer must still hold it; ALORA_ESTATE if there was no evaluation).  V, W: DEVICE, ctx
 * dtype, row-major n x p, contiguous (ld = p); p = 1 for vectors.  W must not alias V.
 * vw: HOST double* receiving <V,W> = sum_ij V_ij W_ij (the Lanczos alpha for p = 1), or NULL; the call
 * synchronises only if vw != NULL. */
alora_status alora_smatvec(alora_ctx *ctx, const double *mu_dev, const void *V, int32_t p, void *W,
                           double *vw);

/* CUDA graphs: alora_eval (stats == NULL), alora_linesearch (p == NULL) and alora_smatvec (vw == NULL) only enqueue
 * kernels on the ctx stream -- no synchronisation, no allocation after the first call with the same shapes -- so a
 * sequence of them can be captured into a CUDA graph on that stream and replayed; alora_get_stats /
 * alora_get_linesearch read the results of the last replay. */

/* Measurement hook (bench.py): when enabled, alora_eval brackets its dominant kernel (the fused
 * row pass of the diagonal class, the adjoint pass of the general class) with CUDA events on the ctx
 * stream; alora_kernel_timing_read synchronises, returns the summed kernel time and the number of
 * launches timed since the last read (at most 8192 between reads), and resets.  enable = k > 1 brackets every
 * k-th evaluation only (two event records cost about 5 us of stream time per evaluation). */
alora_status alora_kernel_timing(alora_ctx *ctx, int enable);
alora_status alora_kernel_timing_read(alora_ctx *ctx, double *total_ms, int64_t *count);

/* The p_want smallest Ritz pairs of S(mu) by Lanczos with full re-orthogonalisation (Alg. 1 line 5, PAPER.md:913:
 * "r-many negative smallest eigenvectors", :932-934; readings 9 and 29): start vector
 * v0[i] = counter_uniform(seed, i); the run stops at step k when the SMALLEST pair's residual estimate
 * |beta_k s_k| <= tol_abs, on breakdown, or at k = kmax (then ALORA_ENOTCONV with the best pairs so far); the
 * min(p_want, k) smallest Ritz pairs of that k-step tridiagonal are returned (a Ritz vector's Rayleigh quotient
 * is its Ritz value whether or not the pair has converged; resid says how far each one is).
 * mu_dev: DEVICE fp64[m], or NULL = lambda of the last alora_eval (as in alora_smatvec).  1 <= p_want <= 8.
 * theta: HOST double[p_want], ascending.  V_dev: DEVICE, ctx dtype, p_want vectors of length n, COLUMN-major
 * (unit Ritz vector j is the contiguous array V_dev + j*n), or NULL.  p_found: HOST int32* (pairs returned);
 * k_used: HOST int32* (Lanczos steps); resid: HOST double[p_want] (|beta_k s_{k,j}| per pair).  theta, p_found,
 * k_used, resid may each be NULL.  Synchronises. */
alora_status alora_lanczos(alora_ctx *ctx, const double *mu_dev, int32_t kmax, double tol_abs, uint64_t seed,
                           int32_t p_want, double *theta, void *V_dev, int32_t *p_found, int32_t *k_used,
                           double *resid);

/* Free constants of the ALORA loop (Algorithm 1; readings in DESIGN.md).  Fill with
 * alora_default_params, then edit. */
typedef struct {
  double eps;          /* KKT tolerance of eq. 77 (1e-5) */
  int32_t stop_mode;   /* 0: all three terms of eq. 77 <= eps;  1: primal infeasibility term only */
  int32_t T_max;       /* outer iterations (100) */
  double tol0, c_in, tol_min; /* inner tolerance tol_t = max(tol_min, min(tol0, c_in*infeas_{t-1})): 1e-2, 0.1, 1e-7 */
  int32_t it_max;      /* inner iterations per outer iteration (500) */
  int32_t lbfgs_mem;   /* L-BFGS pairs (5), at most 16 (larger values are clamped to 16); 0 = steepest descent with the exact step */
  int32_t p_max;       /* eigenvectors per growth step, 1..4 (1: closed-form step; more: every sufficiently negative
                          Ritz pair of the Lanczos run, small SDP of Alg. 1 line 7; reading 29) */
  int32_t k_max;       /* Lanczos steps (300) */
  double tau_neg;      /* growth threshold on -theta_1/(1+||C||_F); < 0 means eps */
  double tol_eig;      /* Lanczos residual tolerance relative to (1+||C||_F); < 0 means eps/10 */
  double gamma, kappa, sigma_max; /* sigma <- min(gamma sigma, sigma_max) if ||q|| > kappa ||q_prev||: 2, 0.25, 1e8 */
  double tau_shrink;   /* drop directions of R^T R with mu_j <= tau_shrink*mu_max (1e-8) */
  double s_max;        /* cap of the growth step when A(vv^T) = 0 (1e6) */
  uint64_t seed;       /* Lanczos start vectors use seed + run index (12345) */
  double stall_tol;    /* inner loop also stops after stall_iters consecutive steps whose predicted decrease
                          phi(0) - phi(alpha) is <= stall_tol * (1 + |f|)  (0 = off, the default; reading 28) */
  int32_t stall_iters; /* (3) */
  int32_t pad_;
} alora_params;
void alora_default_params(alora_params *p);
/* Defaults adjusted to the context dtype.  ALORA_F64: alora_default_params.  ALORA_F32: the gradient norm of an fp32
 * evaluation cannot fall below its rounding floor, so late outer iterations would spend all it_max = 500 inner
 * iterations without decreasing f; the preset bounds the inner solves -- "approximately solving" the subproblem is
 * what the paper's practical variant does -- with it_max = 100 and the stall rule on
 * (stall_tol = 1e-9, stall_iters = 3; readings 6 and 28).  oracle/alm.py has the same preset. */
void alora_preset_params(alora_params *p, alora_dtype dtype);

typedef struct { /* one row per outer iteration */
  int32_t t, r, inner_iters, n_evals, lanczos_steps, grew, shrank, pad_;
  double sigma, cx, f, qnorm, gnorm, theta1, kkt[3];
} alora_iter_record;

typedef struct {
  int32_t converged, outer_iters, n_evals, n_linesearch, n_matvec, r_final;
  double kkt[3], sigma_final, seconds;
} alora_result;

/* ALORA (Algorithm 1) on the ctx's problem.  State in/out: R_dev (DEVICE, ctx dtype, capacity
 * n*r_cap elements; on entry row-major n x *r_inout with ld = *r_inout, on exit row-major
 * n x *r_inout with ld = *r_inout), y_dev (DEVICE fp64[m], updated in place), *sigma_inout.
 * r_cap bounds the rank: an outer iteration that would grow beyond it skips the growth step and carries on
 * at rank r_cap (reading 27).  log: HOST array of log_cap records or NULL.
 * Returns ALORA_OK on convergence, ALORA_ENOTCONV at T_max.  (R, r, y, sigma) is the whole state of
 * Alg. 1, so a caller can checkpoint / resume with it. */
alora_status alora_solve(alora_ctx *ctx, const alora_params *prm, void *R_dev, int32_t *r_inout,
                         int32_t r_cap, double *y_dev, double *sigma_inout, alora_iter_record *log,
                         int32_t log_cap, alora_result *res);

#ifdef __cplusplus
}
#endif
#endif /* ALORA_H */
