/* oracle/pdbo_oracle.c -- CPU ORACLE for PDBO (arxiv 2509.21064).  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct implementation of what the hot path computes, written from
 * /root/reference/PAPER.md and the readings R0-R14 listed in DESIGN.md.  It shares no code with the
 * CUDA library; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call it.  No blocking, fusion or reordering beyond what the paper states.
 *
 * Precision: compile with -DREAL=double (default; per-step truth) or -DREAL=float (trajectory tests,
 * reading R12).  Exact objective values F(x_hat) are always accumulated in double.
 *
 * Parity pins (tests/test_oracle_pins.py): F by brute force and edge list; f by Def. 2.2 enumeration;
 * grad f by multilinearity; the Max-Cut fixed point at 1/2; Hessian 2(W+diag y)
 * (PAPER.md:606); step invariants; convex special case; 2^20 brute force;
 * PDBO-s: finite differences of L_s in x and mu, n = 1 equals PDBO, the multiplier stays one number per restart.
 * Unpinned: optimality of the objective reached on configs 2-5 (no optimum known) -- see DESIGN.md.
 *
 * Layout: iterates are [n][B] row-major (restart index contiguous), as at the library's C ABI.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef REAL
#define REAL double
#endif
typedef REAL real;
#define NEXT_AFTER(a, b) (sizeof(real) == 4 ? (double)nextafterf((float)(a), (float)(b)) : nextafter((double)(a), (double)(b)))

#define KIND_QUBO_CSR 0
#define KIND_QUBO_DENSE 1
#define KIND_MAXSAT 2
#define G_QUADRATIC 0
#define G_ENTROPY 1
#define DUAL_PER_VARIABLE 0
#define DUAL_SCALAR 1

/* Problem data, all host pointers owned by the caller.
 * QUBO: F(x) = x^T Q x + c^T x for ANY square Q (diagonal and asymmetry allowed here; reading R1).
 * MaxSAT: F(x) = sum_j w_j prod_{l in C_j} p_l(x)  (weights: reading R9). */
typedef struct {
    int32_t kind;
    int32_t n;
    /* KIND_QUBO_CSR: entries (i, col[k], val[k]) for rowptr[i] <= k < rowptr[i+1] */
    const int32_t* rowptr;
    const int32_t* col;
    const double* val;
    /* KIND_QUBO_DENSE: Q row-major [n][n]; Qt = its transpose, also row-major (so that Q_ji is read
     * contiguously: Qt[i*n+j] == Qd[j*n+i]); the Python wrapper fills both */
    const double* Qd;
    const double* Qt;
    const double* c; /* [n] or NULL (= 0), both QUBO kinds */
    /* KIND_MAXSAT: clause j holds literals lit[cptr[j] .. cptr[j+1]), lit = +-(var+1) */
    int32_t m;
    const int32_t* cptr;
    const int32_t* lit;
    const double* w; /* [m] or NULL (= 1) */
} pdbo_problem;

/* ---- binarity function g and its derivative (reading R4) ---------------- */
static real xlogx(real u) { return (u > (real)0) ? u * (real)log((double)u) : (real)0; }

static real g_fun(int gfun, real x) {
    if (gfun == G_QUADRATIC) return x * x - x;                 /* g(x) = x^2 - x        (212) */
    return xlogx(x) + xlogx((real)1 - x);                      /* x ln x + (1-x)ln(1-x) (110) */
}

static real g_prime(int gfun, real x, real eps) {
    if (gfun == G_QUADRATIC) return (real)2 * x - (real)1;
    real xc = x;                                               /* R4: clip to [eps, 1-eps] */
    if (xc < eps) xc = eps;
    if (xc > (real)1 - eps) xc = (real)1 - eps;
    return (real)log((double)xc) - (real)log((double)((real)1 - xc));
}

/* ---- literal term p(x_i) and its derivative sign -------------------------------- */
/* positive literal (lit > 0): p = 1 - x, dp/dx = -1;  negated literal (lit < 0): p = x, dp/dx = +1 */
static int lit_var(int32_t l) { return (l > 0 ? l : -l) - 1; }
static real lit_p(int32_t l, real x) { return l > 0 ? (real)1 - x : x; }
static real lit_s(int32_t l) { return l > 0 ? (real)-1 : (real)1; }

/* ---- gradient of the multilinear extension f for ONE restart column (contiguous x[n]) ----------- */
/* QUBO (Prop. 2.4 with x_i^2 -> x_i, reading R1): f(x) = sum_{i!=j} Q_ij x_i x_j + sum_i (Q_ii + c_i) x_i
 *   d f / d x_i = sum_{j != i} (Q_ij + Q_ji) x_j + Q_ii + c_i.
 * MaxSAT: d/dx_i of w_j prod_l p_l = w_j * s_i * prod_{l != i} p_l   (leave-one-out product, no division). */
static void grad_f(const pdbo_problem* P, const real* x, real* G) {
    const int n = P->n;
    for (int i = 0; i < n; ++i) G[i] = (P->kind != KIND_MAXSAT && P->c) ? (real)P->c[i] : (real)0;
    if (P->kind == KIND_QUBO_CSR) {
        for (int i = 0; i < n; ++i)
            for (int k = P->rowptr[i]; k < P->rowptr[i + 1]; ++k) {
                const int j = P->col[k];
                const real q = (real)P->val[k];
                if (j == i) { G[i] += q; }
                else { G[i] += q * x[j]; G[j] += q * x[i]; }   /* Q_ij appears in d/dx_i and d/dx_j */
            }
    } else if (P->kind == KIND_QUBO_DENSE) {
        for (int i = 0; i < n; ++i) {
            real acc = (real)0;
            for (int j = 0; j < n; ++j) {
                if (j == i) continue;
                acc += ((real)P->Qd[(size_t)i * n + j] + (real)P->Qt[(size_t)i * n + j]) * x[j];  /* Q_ij + Q_ji */
            }
            G[i] += acc + (real)P->Qd[(size_t)i * n + i];
        }
    } else {
        for (int j = 0; j < P->m; ++j) {
            const real wj = P->w ? (real)P->w[j] : (real)1;
            for (int a = P->cptr[j]; a < P->cptr[j + 1]; ++a) {
                real prod = (real)1;
                for (int b = P->cptr[j]; b < P->cptr[j + 1]; ++b)
                    if (b != a) prod *= lit_p(P->lit[b], x[lit_var(P->lit[b])]);
                G[lit_var(P->lit[a])] += wj * lit_s(P->lit[a]) * prod;
            }
        }
    }
}

/* ---- multilinear extension f(x), closed form of Prop. 2.4, one column ---------- */
static double f_ext(const pdbo_problem* P, const real* x) {
    const int n = P->n;
    double f = 0.0;
    if (P->kind == KIND_QUBO_CSR) {
        for (int i = 0; i < n; ++i)
            for (int k = P->rowptr[i]; k < P->rowptr[i + 1]; ++k) {
                const int j = P->col[k];
                f += (j == i) ? P->val[k] * (double)x[i] : P->val[k] * (double)x[i] * (double)x[j];
            }
    } else if (P->kind == KIND_QUBO_DENSE) {
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j)
                f += (j == i) ? P->Qd[(size_t)i * n + i] * (double)x[i]
                              : P->Qd[(size_t)i * n + j] * (double)x[i] * (double)x[j];
    } else {
        for (int j = 0; j < P->m; ++j) {
            double prod = P->w ? P->w[j] : 1.0;
            for (int a = P->cptr[j]; a < P->cptr[j + 1]; ++a)
                prod *= (double)lit_p(P->lit[a], x[lit_var(P->lit[a])]);
            f += prod;
        }
        return f;
    }
    if (P->c) for (int i = 0; i < n; ++i) f += P->c[i] * (double)x[i];
    return f;
}

/* ---- exact objective F on a binary point (187-189; 196), one column ------------- */
/* QUBO: x^T Q x + c^T x written out.  MaxSAT: weight of clauses whose literals are all false
 * (a positive literal is false iff x=0, a negated one iff x=1).                                     */
static double F_binary(const pdbo_problem* P, const uint8_t* xh) {
    const int n = P->n;
    double F = 0.0;
    if (P->kind == KIND_QUBO_CSR) {
        for (int i = 0; i < n; ++i) {
            if (!xh[i]) continue;
            for (int k = P->rowptr[i]; k < P->rowptr[i + 1]; ++k)
                if (xh[P->col[k]]) F += P->val[k];
        }
    } else if (P->kind == KIND_QUBO_DENSE) {
        for (int i = 0; i < n; ++i) {
            if (!xh[i]) continue;
            for (int j = 0; j < n; ++j)
                if (xh[j]) F += P->Qd[(size_t)i * n + j];
        }
    } else {
        for (int j = 0; j < P->m; ++j) {
            int all_false = 1;
            for (int a = P->cptr[j]; a < P->cptr[j + 1]; ++a) {
                const int32_t l = P->lit[a];
                const int v = xh[lit_var(l)];
                const int truth = (l > 0) ? v : !v;
                if (truth) { all_false = 0; break; }
            }
            if (all_false) F += P->w ? P->w[j] : 1.0;
        }
        return F;
    }
    if (P->c) for (int i = 0; i < n; ++i) if (xh[i]) F += P->c[i];
    return F;
}

/* ---- perturbation side when both x^t and the tentative iterate sit exactly at 1/2 (reading R3) --- */
/* A written-out 32-bit integer mix of (seed, t, i, b); the CUDA library implements the same integer
 * function on its own.  Returns +1 or -1.                                                            */
static uint32_t mix32(uint32_t h) {
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    return h;
}
static int side_bit(uint64_t seed, uint32_t t, uint32_t i, uint32_t b) {
    uint32_t h = mix32((uint32_t)seed ^ ((uint32_t)(seed >> 32) * 0x9E3779B9u));
    h = mix32(h + t);
    h = mix32(h + i);
    h = mix32(h + b);
    return (h & 1u) ? +1 : -1;
}

typedef struct {
    double alpha, beta;   /* step sizes                      */
    double delta;         /* perturbation band half width, 0 disables (R3)      */
    double log_eps;       /* clamp of g' for the entropy g (R4)                 */
    int32_t gfun;         /* G_QUADRATIC | G_ENTROPY                            */
    int32_t iters;        /* T_max: exactly this many steps (R0)                */
    int32_t eval_every;   /* round + score every this many steps and at the end (R5) */
    int32_t t0;           /* iteration index of x0 (enters the tie-break hash only) */
    uint64_t seed;
    int32_t dual;         /* DUAL_PER_VARIABLE (PDBO, Eq. 6) | DUAL_SCALAR (PDBO-s; reading R14) */
} pdbo_params;

/* ---- one simultaneous projected GDA step, Eq. (6) + perturbation (148, 732) --- */
/* x, y: time-t values (contiguous, one restart).  xn, yn: time-(t+1) values.  G: scratch [n].        */
/* PDBO-s (the single constraint sum_i g(x_i) = 0 with one multiplier mu; reading R14):     */
/*   L_s(x, mu) = f(x) + mu sum_i g(x_i);  x+ = clip(x - alpha (grad f + mu g'(x)));  mu+ = mu + beta sum_i g(x_i) */
/* mu is kept replicated in y[0..n): every entry receives the same increment.                               */
static void gda_step(const pdbo_problem* P, const pdbo_params* hp, uint32_t t, uint32_t b,
                     const real* x, const real* y, real* xn, real* yn, real* G) {
    const int n = P->n;
    const real alpha = (real)hp->alpha, beta = (real)hp->beta, delta = (real)hp->delta;
    const real half = (real)0.5;
    grad_f(P, x, G);
    real gsum = (real)0;                                       /* PDBO-s: grad_mu L_s = sum_i g(x_i^t), index order */
    if (hp->dual == DUAL_SCALAR)
        for (int i = 0; i < n; ++i) gsum += g_fun(hp->gfun, x[i]);
    for (int i = 0; i < n; ++i) {
        const real gp = g_prime(hp->gfun, x[i], (real)hp->log_eps);
        const real gv = g_fun(hp->gfun, x[i]);
        real xt = x[i] - alpha * (G[i] + y[i] * gp);           /* x - alpha * grad_x L          */
        if (xt < (real)0) xt = (real)0;                        /* projection onto [0,1]         */
        if (xt > (real)1) xt = (real)1;
        yn[i] = y[i] + beta * (hp->dual == DUAL_SCALAR ? gsum : gv);   /* y + beta * grad_y L, uses x^t */
        if (delta > (real)0 && fabs((double)(x[i] - half)) < (double)delta
                            && fabs((double)(xt - half)) < (double)delta) {
            int s;                                             /* R3: two successive in-band iterates */
            if (xt > half) s = +1; else if (xt < half) s = -1;
            else if (x[i] > half) s = +1; else if (x[i] < half) s = -1;
            else s = side_bit(hp->seed, t, (uint32_t)i, b);
            xt = half + delta * (real)s;                       /* project onto {|x-1/2| >= delta} */
            if (fabs((double)(xt - half)) < (double)delta)     /* rounding fell inside: step one ulp away  */
                xt = (real)NEXT_AFTER(xt, s > 0 ? (real)2 : (real)-1);   /* so that |x-1/2| >= delta holds */
        }
        xn[i] = xt;
    }
}

/* ---- exported entry points (all arrays [n][B] row-major unless noted) --------------------------- */

/* G = grad f(X) column by column. */
int pdbo_grad(const pdbo_problem* P, int32_t B, const real* X, real* Gout) {
    const int n = P->n;
    real* x = (real*)calloc(n, sizeof(real));
    real* G = (real*)calloc(n, sizeof(real));
    if (!x || !G) return 1;
    for (int b = 0; b < B; ++b) {
        for (int i = 0; i < n; ++i) x[i] = X[(size_t)i * B + b];
        grad_f(P, x, G);
        for (int i = 0; i < n; ++i) Gout[(size_t)i * B + b] = G[i];
    }
    free(x); free(G);
    return 0;
}

/* out[b] = f(X[:,b]) (closed form of Prop. 2.4). */
int pdbo_f(const pdbo_problem* P, int32_t B, const real* X, double* out) {
    const int n = P->n;
    real* x = (real*)malloc(sizeof(real) * n);
    if (!x) return 1;
    for (int b = 0; b < B; ++b) {
        for (int i = 0; i < n; ++i) x[i] = X[(size_t)i * B + b];
        out[b] = f_ext(P, x);
    }
    free(x);
    return 0;
}

/* out[b] = L(X[:,b], Y[:,b]) = f(x) + sum_i y_i g(x_i); the value whose minimum over x, for y
 * with L(., y) convex, is the dual certificate of PAPER.md:1105-1114. */
int pdbo_lagrangian(const pdbo_problem* P, int32_t B, const real* X, const real* Y, int32_t gfun, double* out) {
    const int n = P->n;
    real* x = (real*)malloc(sizeof(real) * n);
    if (!x) return 1;
    for (int b = 0; b < B; ++b) {
        double constraint = 0.0;
        for (int i = 0; i < n; ++i) {
            x[i] = X[(size_t)i * B + b];
            constraint += (double)Y[(size_t)i * B + b] * (double)g_fun(gfun, x[i]);
        }
        out[b] = f_ext(P, x) + constraint;
    }
    free(x);
    return 0;
}

/* out[b] = F(Xh[:,b]) on binary columns. */
int pdbo_F(const pdbo_problem* P, int32_t B, const uint8_t* Xh, double* out) {
    const int n = P->n;
    uint8_t* xh = (uint8_t*)malloc(n);
    if (!xh) return 1;
    for (int b = 0; b < B; ++b) {
        for (int i = 0; i < n; ++i) xh[i] = Xh[(size_t)i * B + b];
        out[b] = F_binary(P, xh);
    }
    free(xh);
    return 0;
}

/* Algorithm 1 (reconstructed, R0) for B independent restarts.
 *   X0, Y0      in : [n][B]
 *   col_ids     in : [B] restart index used in the tie-break hash, or NULL for 0..B-1 (lets a test run
 *                    a subset of the columns of a larger batch)
 *   x_bin       out: [n][B] best-so-far rounded point per restart (R5), may be NULL
 *   obj         out: [B] its objective, may be NULL
 *   best_restart out: argmin_b obj[b], ties -> lowest b (R6), may be NULL
 *   Xf, Yf      out: final iterates [n][B], may be NULL
 *   nthreads       : OpenMP threads over restarts (restarts are independent); <=1 = serial          */
int pdbo_run(const pdbo_problem* P, int32_t B, const real* X0, const real* Y0, const int32_t* col_ids,
             const pdbo_params* hp, uint8_t* x_bin, double* obj, int32_t* best_restart,
             real* Xf, real* Yf, int32_t nthreads) {
    const int n = P->n;
    int fail = 0;
    double* best = (double*)malloc(sizeof(double) * (B > 0 ? B : 1));
    if (!best) return 1;
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
#endif
    for (int b = 0; b < B; ++b) {
        real* x = (real*)malloc(sizeof(real) * n);
        real* y = (real*)malloc(sizeof(real) * n);
        real* xn = (real*)malloc(sizeof(real) * n);
        real* yn = (real*)malloc(sizeof(real) * n);
        real* G = (real*)malloc(sizeof(real) * n);
        uint8_t* xh = (uint8_t*)malloc(n);
        uint8_t* bx = (uint8_t*)calloc(n, 1);
        if (!x || !y || !xn || !yn || !G || !xh || !bx) { fail = 1; }
        else {
            const uint32_t bid = col_ids ? (uint32_t)col_ids[b] : (uint32_t)b;
            double bv = INFINITY;
            for (int i = 0; i < n; ++i) { x[i] = X0[(size_t)i * B + b]; y[i] = Y0[(size_t)i * B + b]; }
            for (int t = 0; t < hp->iters; ++t) {
                gda_step(P, hp, (uint32_t)(hp->t0 + t), bid, x, y, xn, yn, G);
                real* tmp = x; x = xn; xn = tmp;
                tmp = y; y = yn; yn = tmp;
                if ((t + 1) % hp->eval_every == 0 || t == hp->iters - 1) {
                    for (int i = 0; i < n; ++i) xh[i] = (x[i] > (real)0.5) ? 1 : 0;   /* R5 */
                    const double v = F_binary(P, xh);
                    if (v < bv) { bv = v; memcpy(bx, xh, n); }
                }
            }
            best[b] = bv;
            if (obj) obj[b] = bv;
            if (x_bin) for (int i = 0; i < n; ++i) x_bin[(size_t)i * B + b] = bx[i];
            if (Xf) for (int i = 0; i < n; ++i) Xf[(size_t)i * B + b] = x[i];
            if (Yf) for (int i = 0; i < n; ++i) Yf[(size_t)i * B + b] = y[i];
        }
        free(x); free(y); free(xn); free(yn); free(G); free(xh); free(bx);
    }
    if (best_restart && !fail) {
        int arg = 0;
        for (int b = 1; b < B; ++b) if (best[b] < best[arg]) arg = b;      /* ties -> lowest b (R6) */
        *best_restart = arg;
    }
    free(best);
    return fail;
}

int pdbo_sizeof_real(void) { return (int)sizeof(real); }
int pdbo_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
int pdbo_side_bit(uint64_t seed, uint32_t t, uint32_t i, uint32_t b) { return side_bit(seed, t, i, b); }
