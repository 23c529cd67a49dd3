/* include/gda.h -- C ABI of the B200-native GDA hot path of PDBO (arxiv 2509.21064).
 *
 * The library solves   min_{x in {0,1}^n} F(x)   (Eq. 1) by simultaneous projected
 * gradient descent-ascent (Eq. 6) on the Lagrangian
 *     L(x, y) = f(x) + sum_i y_i g(x_i)
 * of the multilinear extension f of F (Def. 2.2, 69-73 Prop. 2.4), for B independent
 * restarts at once, with periodic rounding, exact scoring and an arg-best over
 * restarts.  The dual variable the paper calls y is `lambda` here.
 *
 * Conventions
 *   - Plain C, no exceptions or aborts across the boundary; every entry point returns a gda_status and
 *     leaves a thread-local message for gda_last_error().  `out` handles are NULL on failure.
 *   - "HOST" / "DEVICE" says where a pointer must live.  The library never frees or keeps caller memory
 *     (problem data is copied at create).
 *   - Iterates are fp32, layout [n][B] row-major: element (variable i, restart b) at i*B + b, so the
 *     restart index is contiguous.  Any B >= 1 is served (the paper runs B = 1, 10, 100, 1000: PAPER.md:836-843, 873-878):
 *     the kernels work on 128-bit vectors of 4 restarts, so inside its workspace the library pads the restart axis with
 *     zero-initialised restarts up to a multiple of 4 (dense problems: 128; sometimes 8 for B <= 64, so that a row is whole
 *     32-byte sectors) that run along and are never read -- not by
 *     the evaluation, the trace, the arg-best or the copies out.  When the row stride differs from B, gda_grad / gda_score / gda_lagrangian go
 *     through zero-padded copies in the workspace (and, like dense problems always, invalidate a state to resume from).
 *   - gda_run / gda_grad / gda_score enqueue work on `stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) and return without synchronising; outputs are valid once the stream has
 *     reached that point.  A handle must not be used from two streams or threads at the same time; different
 *     handles may be used from different host threads concurrently.
 *   - All compute runs in CUDA kernels for sm_100a; there is no CPU fallback: without a usable device
 *     every compute entry point fails with GDA_ERR_CUDA.
 */
#ifndef GDA_H_
#define GDA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gda_problem gda_problem; /* opaque; owns the device copies of the problem and a workspace */

typedef enum {
    GDA_OK = 0,
    GDA_ERR_INVALID_ARG = 1, /* null pointer, bad size, asymmetric Q, index out of range, bad parameter ... */
    GDA_ERR_ALLOC = 2,       /* host or device allocation failed */
    GDA_ERR_CUDA = 3,        /* a CUDA call or kernel launch failed (message has the CUDA error string) */
    GDA_ERR_UNSUPPORTED = 4  /* valid request this build cannot serve (e.g. a dense problem without GDA_DENSE_BF16) */
} gda_status;

/* binarity function g (default quadratic; entropy for Max-k-SAT, 580/592) */
typedef enum {
    GDA_G_QUADRATIC = 0, /* g(x) = x^2 - x,                     g'(x) = 2x - 1                      */
    GDA_G_ENTROPY = 1    /* g(x) = x ln x + (1-x) ln(1-x), 0 at the ends; g'(x) = ln(xc) - ln(1-xc),
                            xc = clip(x, log_eps, 1-log_eps)   (reading R4)               */
} gda_gfun;

#define GDA_DENSE_BF16 1 /* gda_create_qubo_dense flag: store Q in bf16, fp32 accumulate (tcgen05 path) */

/* ---- problems ---------------------------------------------------------------------------------------
 * QUBO: F(x) = x^T Q x + c^T x.  Q must be symmetric.  A non-zero diagonal is folded into
 * the linear term, f(x) = sum_{i!=j} Q_ij x_i x_j + sum_i (Q_ii + c_i) x_i  (Prop. 2.4 with x_i^2 -> x_i;
 * DESIGN.md reading R1).  Max-Cut with weight matrix W is Q = W, c = -W 1 and
 * cut(x) = -F(x).
 *
 * gda_create_qubo_csr: HOST rowptr[n+1], col[nnz], val[nnz] (both (i,j) and (j,i) stored, any order within
 *   a row, no duplicate (i,j)), HOST c[n] or NULL (= 0).
 *   INVALID_ARG: n <= 0, null pointers, rowptr not non-decreasing from 0, column out of range, duplicate
 *   entry, Q_ij != Q_ji, non-finite value. */
gda_status gda_create_qubo_csr(int32_t n, const int32_t* rowptr, const int32_t* col, const float* val,
                               const float* c, gda_problem** out);

/* gda_create_qubo_dense: HOST Q row-major [n][n] (symmetric), HOST c[n] or NULL.  flags must contain
 *   GDA_DENSE_BF16: Q is rounded to bf16 (lossless when Q is bf16-representable, reading R13)
 *   and the gradient is a tcgen05 GEMM with fp32 accumulation.  UNSUPPORTED: flags without GDA_DENSE_BF16.
 *   Any n > 0 and any B > 0 are served: internally n is zero-padded to a multiple of 256 and B to a
 *   multiple of 128 (the GEMM tile), which costs the padded work but changes no result. */
gda_status gda_create_qubo_dense(int32_t n, const float* Q, const float* c, int32_t flags, gda_problem** out);

/* Weighted MaxSAT: F(x) = sum_j w_j [clause j unsatisfied] = sum_j w_j prod_{l in C_j} p_l(x)
 * (weights: DESIGN.md reading R9).  HOST cptr[m+1], lit[cptr[m]] with
 * lit = +(var+1) for a positive literal (p = 1 - x) and -(var+1) for a negated one (p = x), HOST w[m] or
 * NULL (= all 1).  Weights may have either sign: the same entry point then minimises ANY polynomial given as a sum of
 * weighted literal products over distinct variables (Prop. 2.4, is stated for polynomials) -- a monomial
 * a prod_{i in S} x_i is the clause of the negated literals of S with weight a, and the indicator of a joint assignment of
 * a clique (the terms of MAP inference on a binary MRF) is the clause that assignment falsifies.
 * INVALID_ARG: empty clause, variable out of range, a variable repeated inside one clause (the product would not be the
 * multilinear extension, reading R2), non-finite weight.  UNSUPPORTED: a clause of more than 65 literals. */
gda_status gda_create_maxsat(int32_t n, int32_t m, const int32_t* cptr, const int32_t* lit, const float* w,
                             gda_problem** out);

/* Max-k-Cut (Appendix B): minimise Tr(X W X^T) over X in R^{k x n} with one-hot columns, i.e.
 * maximise the weight of the edges between different parts, cut = (sum_ij W_ij - obj) / 2.  HOST CSR of the
 * SYMMETRIC weight matrix W (both directions stored), 2 <= k <= 8.  The method runs on logits Z with
 * X_{:,i} = SoftMax(Z_{:,i}) (readings K1-K5), so for such a problem gda_run takes
 *   x0           DEVICE fp32 [k][n][B]: the initial logits Z^0
 *   lambda0      DEVICE fp32 [n][B] or NULL (lambda0_scalar)
 *   x_bin        DEVICE uint8 [n][B]: per restart the LABELS (argmax_j Z_ji, lowest j on ties) of the best evaluation
 *   obj          DEVICE double [B]: Tr(Xh W Xh^T) of those labels (exact integers for integer weights)
 *   extra->x_final [k][n][B] logits Z^T; params->delta is ignored (no perturbation is described for this variant);
 *   params->dual must be GDA_DUAL_PER_VARIABLE.  gda_grad / gda_score / gda_lagrangian take the logits (see there).
 * INVALID_ARG: as gda_create_qubo_csr, plus a non-zero diagonal entry and k outside [2, 8]. */
gda_status gda_create_maxkcut(int32_t n, int32_t k, const int32_t* rowptr, const int32_t* col, const float* val,
                              gda_problem** out);

void gda_destroy(gda_problem* p); /* NULL-safe; waits for the work this handle has enqueued, then frees.  (It does not
                                     call cudaDeviceSynchronize: other handles may be capturing on other threads.) */

/* ---- the run ----------------------------------------------------------------------------------------- */
/* Dual variables.  GDA_DUAL_PER_VARIABLE is the paper's method, one multiplier y_i per constraint g(x_i) = 0
 * (Eq. 6).  GDA_DUAL_SCALAR is the ablation "PDBO-s": the single
 * constraint sum_i g(x_i) = 0 with one multiplier mu per restart,
 *     x+ = clip(x - alpha (grad f(x) + mu g'(x))),   mu+ = mu + beta sum_i g(x_i)      (reading R14)
 * the sum accumulated in fp32 in a fixed order (deterministic).  In this mode lambda0 and lambda_final are
 * DEVICE fp32 [B] (HOST [B] for gda_run_host).  Not for Max-k-Cut problems (UNSUPPORTED). */
typedef enum { GDA_DUAL_PER_VARIABLE = 0, GDA_DUAL_SCALAR = 1 } gda_dual;

typedef struct {
    float alpha;        /* primal step size > 0                                          */
    float beta;         /* dual step size >= 0; 0 keeps the multipliers fixed   */
    float delta;        /* perturbation band half-width in [0, 1/2); 0 disables (R3) */
    float log_eps;      /* clamp for g' of the entropy g, in (0, 1/2) (R4); ignored for the quadratic g */
    int32_t iters;      /* T_max >= 0: exactly this many GDA steps (R0)                                 */
    int32_t eval_every; /* > 0: round + score every eval_every steps and after the last step (R5)       */
    int32_t gfun;       /* gda_gfun                                                                     */
    int32_t t0;         /* iteration index of x0 (only enters the exact-1/2 tie-break hash, R3)         */
    uint64_t seed;      /* seed of that hash                                                            */
    int32_t dual;       /* gda_dual: per-variable multipliers (PDBO) or one per restart (PDBO-s)        */
    int32_t reserved;   /* must be 0                                                                    */
} gda_params;

/* Optional extra outputs of gda_run; every pointer is DEVICE memory and may be NULL. */
typedef struct {
    float* x_final;       /* [n][B] iterate x^T                                                         */
    float* lambda_final;  /* [n][B] dual iterate y^T  ([B] with GDA_DUAL_SCALAR)                        */
    double* best_obj;     /* [1]    obj[best_restart]                                                   */
    double* trace_best;   /* [trace_cap] min over restarts of the best objective after evaluation k     */
    uint64_t* trace_ns;   /* [trace_cap] GPU globaltimer (ns) when evaluation k finished                */
    int32_t trace_cap;    /* entries available in the two trace arrays (evaluations beyond it are dropped).  The arrays   *
                           * receive the evaluations of THIS call, entry 0 = its first one, also when the call resumes *
                           * an earlier run; one call records at most 4096 evaluations, later ones are not traced, and  *
                           * entries past the call's last evaluation are left as the caller had them                   */
    int32_t* ones;        /* [B]    number of ones in x_bin[:, b].  With obj it decides feasibility where the     *
                           *        objective is a penalised count, e.g. MIS as a QUBO:      *
                           *        F = -|S| + lam * (edges inside S), so S is independent iff obj[b] == -ones[b] */
} gda_extra;

/* Algorithm 1 (reconstructed in DESIGN.md reading R0) for B restarts.
 *   x0          DEVICE fp32 [n][B], values in [0,1]           (x0 ~ U[0,1]^n); or NULL to RESUME:
 *               continue from the iterates, duals, iteration counter and best-so-far that the previous
 *               gda_run on this handle (same B) left in it -- lambda0 and params->t0 are then ignored
 *   lambda0     DEVICE fp32 [n][B] ([B] with GDA_DUAL_SCALAR) or NULL -> every entry = lambda0_scalar (y-bar)
 *   x_bin       DEVICE uint8 [n][B]: per restart, the rounded point x_hat = [x > 1/2] with the best
 *               objective seen at any evaluation (R5)
 *   obj         DEVICE double [B]: F(x_bin[:,b]) -- exact integers when all coefficients are integers
 *   best_restart DEVICE int32 [1]: argmin_b obj[b], ties -> lowest b (R6)
 * UNSUPPORTED: n * B >= 2^30 elements, counted on the padded workspace (B rounded up to a multiple of 4, sometimes 8; dense
 * problems: n to a multiple of 256 and B to a multiple of 128; times k for Max-k-Cut) -- the message prints those sizes.
 * INVALID_ARG: null required pointer, B <= 0, alpha <= 0, beta < 0 or non-finite, delta outside
 * [0, 1/2), eval_every <= 0, iters < 0, unknown gfun or dual, log_eps outside (0, 1/2) with the entropy g;
 * a resumed run (x0 == NULL) whose `dual` differs from the run it continues.                              */
gda_status gda_run(gda_problem* p, int32_t B, const float* x0, const float* lambda0, float lambda0_scalar,
                   const gda_params* params, uint8_t* x_bin, double* obj, int32_t* best_restart,
                   const gda_extra* extra, void* stream);

/* Same run with HOST buffers (x0, lambda0, x_bin, obj, best_restart on the host; `extra` must be NULL):
 * copies the inputs to the device, runs, copies the three results back and synchronises `stream`. */
gda_status gda_run_host(gda_problem* p, int32_t B, const float* x0, const float* lambda0, float lambda0_scalar,
                        const gda_params* params, uint8_t* x_bin, double* obj, int32_t* best_restart,
                        void* stream);

/* ---- single steps of the path, exposed for parity tests and profiling ---------------------------------
 * gda_grad:  G = grad f(X), DEVICE fp32 [n][B] in and out (S1 sparse / S2 dense / S3 MaxSAT of DESIGN.md).
 *            Max-k-Cut: X is the logits Z [k][n][B] and G [k][n][B] = grad_Z Tr(X W X^T) at X = SoftMax(Z), i.e.
 *            X_ji (D_ji - sum_l X_li D_li) with D = 2 X W (the y = 0 part of the step, reading K1).
 * gda_score: obj[b] = F(x_hat), x_hat = [X[:,b] > 1/2]; DEVICE fp32 X [n][B], DEVICE double obj[B] (S5).
 *            Max-k-Cut: X is the logits [k][n][B], scored by their labels argmax_j Z_ji (lowest j on ties).
 * On a DENSE or Max-k-Cut problem (and whenever the row stride differs from B) they and gda_lagrangian use the handle's run
 * state as scratch: a later gda_run must pass x0. */
gda_status gda_grad(gda_problem* p, int32_t B, const float* x, float* G, void* stream);
gda_status gda_score(gda_problem* p, int32_t B, const float* x, double* obj, void* stream);

/* gda_lagrangian: out[b] = L(X[:,b], Y[:,b]) = f(x) + sum_i y_i g(x_i) at a CONTINUOUS point:
 * f is the multilinear extension, products in fp32, sums in fp64.  DEVICE fp32 X [n][B] in [0,1];
 * lambda DEVICE fp32 [n][B] or NULL -> every y_i = lambda_scalar; gfun / log_eps as in gda_params; DEVICE double out[B].
 * This is the value behind the dual certificate of PAPER.md:1105-1114: for y with f_y = L(., y) convex (Max-Cut:
 * y_i >= -lambda_min(W)), run gda_run with beta = 0 (the multipliers stay at lambda0) until x has converged; then
 * out[b] <= min F, i.e. -out[b] is an upper bound on the maximum cut.  Dense problems: f comes from the tcgen05
 * gradient, f = sum_i x_i (G_i + c'_i) / 2, i.e. with the bf16 operand's error (reading R13).  Max-k-Cut: X is the logits Z [k][n][B] and
 * out[b] = L(SoftMax(Z), y) = Tr(X W X^T) + sum_i y_i g(X_:,i) with g of a column as in PAPER.md:802-806 (log_eps unused). */
gda_status gda_lagrangian(gda_problem* p, int32_t B, const float* x, const float* lambda, float lambda_scalar,
                          int32_t gfun, float log_eps, double* out, void* stream);

/* ---- scoring without any allocation -------------------------------------------------------------------
 * gda_score_qubo_csr_static: obj[b] = F(x_hat_b) = x_hat^T Q x_hat + c^T x_hat, x_hat = [X[:,b] > 1/2] (the
 * rounding and scoring step S5, reading R5) -- the result gda_score gives on a gda_create_qubo_csr handle,
 * for callers that must not allocate device memory.
 *
 * Who that is.  A gda_problem handle is cudaMalloc'd memory (problem copy, iterates, a table of partial sums).  A host
 * application that gave its whole HBM to its own pool at start-up, that runs under a latency bound (cudaMalloc / cudaFree may
 * synchronise the whole device and so stall every stream of the process), or that may only touch buffers it was handed,
 * cannot create one.  This entry point needs no handle: the problem is passed as the CSR the caller already keeps on the
 * device, and the partial-sum table lives in a fixed 4 MiB array inside the library's image (GDA_STATIC_SCRATCH_BYTES; a
 * file-scope __device__ array in csrc/gda_static.cu).  It calls no cudaMalloc, cudaFree or other allocating routine.
 *
 * Arguments -- ALL pointers are DEVICE memory of the current device, owned by the caller, nothing is copied or kept:
 *   rowptr int32 [n+1], col int32 [rowptr[n]], val fp32 [rowptr[n]]: Q in CSR, every stored entry (i, j, Q_ij) counted once,
 *          so a symmetric Q has both directions stored; diagonal entries are allowed (x_hat_i^2 = x_hat_i);
 *   c      fp32 [n] or NULL (= 0);   x fp32 [n][B] row-major, any B >= 1 (no alignment needed);   obj double [B], written.
 *   The CSR is NOT validated (that would need a copy to the host): rowptr must be non-decreasing from 0 and every column in
 *   [0, n).  Sums are taken in fp64 in CSR order: exact for integer coefficients.
 * Limits and sharing:
 *   - B <= GDA_STATIC_SCORE_MAX_B (4096), any n > 0.  More restarts: GDA_ERR_UNSUPPORTED (score them in slices of <= 4096).
 *   - every GPU that loads the library holds the 4 MiB until the process exits;
 *   - the array is shared by ALL calls on a GPU.  Calls on one stream are ordered and fine; two calls that overlap on the
 *     GPU (different streams or threads) race on it and return wrong objectives without an error -- serialise them.  It keeps
 *     the previous call's contents; each call overwrites every entry it reads, so nothing needs clearing in between.
 *   - the FIRST call on each GPU looks the array's device address up (cudaGetSymbolAddress, with that GPU current) and may
 *     trigger the load of the module: make it once at start-up, before any stream capture begins.
 *   - the device that `stream` belongs to must be the current device.  Asynchronous on `stream` like gda_score.
 * INVALID_ARG: null pointer (c excepted), n <= 0, B <= 0, a pointer that is not device (or managed) memory.
 * UNSUPPORTED: B > GDA_STATIC_SCORE_MAX_B.  ERR_CUDA: no usable device, or a failed CUDA call. */
#define GDA_STATIC_SCORE_MAX_B 4096
#define GDA_STATIC_SCRATCH_BYTES (4 * 1024 * 1024)
gda_status gda_score_qubo_csr_static(int32_t n, const int32_t* rowptr, const int32_t* col, const float* val,
                                     const float* c, int32_t B, const float* x, double* obj, void* stream);

/* ---- launch options, per handle -----------------------------------------------------------------------
 * The library picks its launch path from the sizes (cost models in csrc/); these switches override a choice for ONE handle,
 * for tests and A/B timing.  No result changes beyond rounding order (the tests compare the paths bit for bit where the
 * arithmetic is the same).  There is no process-wide state: no environment variable is read by the library.  A change takes
 * effect at the next call on the handle (the graphs it has captured are dropped); like every call on a handle it must not
 * run concurrently with another call on the same handle.  INVALID_ARG: null handle, unknown key, value out of range. */
typedef enum {
    GDA_OPT_SPARSE_PATH = 0,    /* sparse QUBO: 0 cost model (default), 1 slab kernel (state in shared memory, whole chunk in one
                                   launch) whenever the instance fits it, 2 streaming kernels (one launch per step)          */
    GDA_OPT_SPLIT_ALL_ROWS = 1, /* sparse QUBO, Max-k-Cut: -1 by the rule (default), 0 a warp per row, 1 every row split      */
    GDA_OPT_NARROW_SPLIT = 2,   /* sparse QUBO, B <= 64: 1 lane groups share long rows (default), 0 one group per row         */
    GDA_OPT_MAXSAT_NARROW = 3,  /* MaxSAT, B <= 64: 1 lane groups share the slots of a variable (default), 0 off               */
    GDA_OPT_DENSE_SHAPE = 4,    /* dense QUBO: -1 the cluster shape the cost model picks (default); 0 one CTA per tile, 1 CTA
                                   pairs, 2 clusters of 2 pairs, 3 clusters of 4 pairs -- at most this shape, sizes permitting */
    GDA_OPT_GRAPHS = 5,         /* 1 replay CUDA graphs of whole chunks (default), 0 enqueue the same kernels directly         */
    GDA_OPT_ROW_GROUPING = 6    /* sparse PDBO-s step: 1 rows walked grouped by adjacency (default), 0 in index order          */
} gda_option;
gda_status gda_set_option(gda_problem* p, int32_t key, int32_t value);

/* ---- queries ------------------------------------------------------------------------------------------ */
typedef struct {
    int32_t kind;        /* 0 sparse QUBO, 1 dense QUBO, 2 MaxSAT, 3 Max-k-Cut                          */
    int32_t n;
    int64_t nnz;         /* off-diagonal non-zeros (sparse), n*n (dense), literals (MaxSAT)             */
    int32_t m;           /* clauses (MaxSAT), else 0                                                    */
    int32_t integral;    /* 1 when every coefficient is an integer: objectives are accumulated in int64 */
    int64_t last_run_kernel_launches; /* kernels launched by the most recent gda_run on this handle     */
    int64_t last_run_step_launches;   /* of those, launches of the per-step kernel                      */
} gda_info;
gda_status gda_get_info(const gda_problem* p, gda_info* info);

const char* gda_last_error(void); /* thread-local message of the last non-OK status ("" if none) */
const char* gda_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GDA_H_ */
