/* oracle/kcut_oracle.c -- CPU ORACLE for PDBO on Max-k-Cut (arxiv 2509.21064, Appendix B).  TEST INFRASTRUCTURE ONLY.
 *
 * Plain loops, one restart at a time, written from /root/reference/PAPER.md:784-828 and the readings K1-K5 of
 * DESIGN.md.  Shares no code with the CUDA library; same rules of use as pdbo_oracle.c.
 *
 *   min_X Tr(X W X^T),  X in R^{k x n}, every column one-hot
 *   X_{:,i} = SoftMax(Z_{:,i}),  L(Z, y) = Tr(X W X^T) + sum_i y_i g(X_{:,i})
 *   g(v) = sum_j v_j^2 - 1 (quadratic)  |  sum_j v_j log v_j (entropy)
 *   GDA "as in Section 3.2":  Z+ = Z - alpha grad_Z L,  y+ = y + beta g(X_{:,i})   (K1)
 *
 * Parity pins (tests/test_kcut_oracle_pins.py): the objective against the edge list over all k^n labelings; k = 2 against
 * the Max-Cut QUBO evaluator; grad_Z L against finite differences of L typed out in the test; conservation of
 * sum_j Z_ji (the softmax Jacobian annihilates constants); y non-increasing; a whole run against brute force;
 * kcut_lagrangian_batch against the same typed-out L and against the objective at one-hot points; kcut_grad_batch
 * against finite differences of that L with y = 0.
 *
 * Layout: Z, X are [k][n][B] row-major (restart index contiguous), y and the labels [n][B].
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

#define G_QUADRATIC 0
#define G_ENTROPY 1

typedef struct {
    int32_t n, k;
    const int32_t* rowptr; /* CSR of the symmetric weight matrix W, zero diagonal, both directions stored */
    const int32_t* col;
    const double* val;
} kcut_problem;

typedef struct {
    double alpha, beta, log_eps;
    int32_t gfun, iters, eval_every;
} kcut_params;

/* X_{:,i} = SoftMax(Z_{:,i}), computed with the maximum subtracted */
static void softmax_cols(int n, int k, const real* z, real* x) {
    for (int i = 0; i < n; ++i) {
        real m = z[i];
        for (int j = 1; j < k; ++j) if (z[(size_t)j * n + i] > m) m = z[(size_t)j * n + i];
        real s = (real)0;
        for (int j = 0; j < k; ++j) { x[(size_t)j * n + i] = (real)exp((double)(z[(size_t)j * n + i] - m)); s += x[(size_t)j * n + i]; }
        for (int j = 0; j < k; ++j) x[(size_t)j * n + i] /= s;
    }
}

static real g_col(int gfun, int n, int k, const real* x, int i) {
    real s = (real)0;
    for (int j = 0; j < k; ++j) {
        const real v = x[(size_t)j * n + i];
        if (gfun == G_QUADRATIC) s += v * v;
        else if (v > (real)0) s += v * (real)log((double)v);   /* 0 log 0 = 0 */
    }
    return gfun == G_QUADRATIC ? s - (real)1 : s;
}

/* Tr(Xh W Xh^T) for a labeling: sum over stored entries (i, l) with equal labels of W_il */
static double kcut_objective(const kcut_problem* P, const uint8_t* lab) {
    double s = 0.0;
    for (int i = 0; i < P->n; ++i)
        for (int a = P->rowptr[i]; a < P->rowptr[i + 1]; ++a)
            if (lab[i] == lab[P->col[a]]) s += P->val[a];
    return s;
}

/* one GDA step for one restart (z, x = softmax(z), y at time t -> zn, yn) */
static void kcut_step(const kcut_problem* P, const kcut_params* hp, const real* z, const real* x, const real* y,
                      real* zn, real* yn, real* D) {
    const int n = P->n, k = P->k;
    const real alpha = (real)hp->alpha, beta = (real)hp->beta;
    for (int i = 0; i < n; ++i) {
        /* D_j = dL/dX_ji = ((W + W^T) X^T)_ij + y_i dg/dX_ji   (W symmetric: 2 (X W)_ji) */
        for (int j = 0; j < k; ++j) {
            real s = (real)0;
            for (int a = P->rowptr[i]; a < P->rowptr[i + 1]; ++a)
                s += (real)2 * (real)P->val[a] * x[(size_t)j * n + P->col[a]];
            const real v = x[(size_t)j * n + i];
            real gp;
            if (hp->gfun == G_QUADRATIC) gp = (real)2 * v;
            else gp = (real)log((double)(v > (real)hp->log_eps ? v : (real)hp->log_eps)) + (real)1;
            D[j] = s + y[i] * gp;
        }
        /* chain rule through the softmax: dL/dZ_ji = X_ji (D_j - sum_l X_li D_l) */
        real mean = (real)0;
        for (int j = 0; j < k; ++j) mean += x[(size_t)j * n + i] * D[j];
        for (int j = 0; j < k; ++j)
            zn[(size_t)j * n + i] = z[(size_t)j * n + i] - alpha * x[(size_t)j * n + i] * (D[j] - mean);
        yn[i] = y[i] + beta * g_col(hp->gfun, n, k, x, i);       /* uses X^t */
    }
}

/* L(SoftMax(Z), y) = Tr(X W X^T) + sum_i y_i g(X_{:,i}) per restart; Z [k][n][B], Y [n][B] */
int kcut_lagrangian_batch(const kcut_problem* P, int32_t B, const real* Z, const real* Y, int32_t gfun, double* out) {
    const int n = P->n, k = P->k;
    const size_t kn = (size_t)k * n;
    real* z = (real*)malloc(sizeof(real) * kn);
    real* x = (real*)malloc(sizeof(real) * kn);
    if (!z || !x) { free(z); free(x); return 1; }
    for (int b = 0; b < B; ++b) {
        for (size_t e = 0; e < kn; ++e) z[e] = Z[e * B + b];
        softmax_cols(n, k, z, x);
        double L = 0.0;
        for (int i = 0; i < n; ++i) {
            for (int j = 0; j < k; ++j) {                        /* Tr(X W X^T) = sum_j sum_{i,l} X_ji W_il X_jl */
                double s = 0.0;
                for (int a = P->rowptr[i]; a < P->rowptr[i + 1]; ++a) s += P->val[a] * (double)x[(size_t)j * n + P->col[a]];
                L += (double)x[(size_t)j * n + i] * s;
            }
            L += (double)Y[(size_t)i * B + b] * (double)g_col(gfun, n, k, x, i);
        }
        out[b] = L;
    }
    free(z); free(x);
    return 0;
}

/* grad_Z of f(SoftMax(Z)) = Tr(X W X^T): dTr/dX_ji = 2 (X W)_ji (W symmetric), then the softmax chain rule
 * d/dZ_ji = X_ji (D_ji - sum_l X_li D_li)  (the y = 0 part of kcut_step).  Z, out [k][n][B] */
int kcut_grad_batch(const kcut_problem* P, int32_t B, const real* Z, real* out) {
    const int n = P->n, k = P->k;
    const size_t kn = (size_t)k * n;
    real* z = (real*)malloc(sizeof(real) * kn);
    real* x = (real*)malloc(sizeof(real) * kn);
    real* D = (real*)malloc(sizeof(real) * k);
    if (!z || !x || !D) { free(z); free(x); free(D); return 1; }
    for (int b = 0; b < B; ++b) {
        for (size_t e = 0; e < kn; ++e) z[e] = Z[e * B + b];
        softmax_cols(n, k, z, x);
        for (int i = 0; i < n; ++i) {
            real mean = (real)0;
            for (int j = 0; j < k; ++j) {
                real s = (real)0;
                for (int a = P->rowptr[i]; a < P->rowptr[i + 1]; ++a) s += (real)2 * (real)P->val[a] * x[(size_t)j * n + P->col[a]];
                D[j] = s;
                mean += x[(size_t)j * n + i] * s;
            }
            for (int j = 0; j < k; ++j) out[((size_t)j * n + i) * B + b] = x[(size_t)j * n + i] * (D[j] - mean);
        }
    }
    free(z); free(x); free(D);
    return 0;
}

int kcut_objective_batch(const kcut_problem* P, int32_t B, const uint8_t* labels, double* out) {
    uint8_t* lab = (uint8_t*)malloc(P->n);
    if (!lab) return 1;
    for (int b = 0; b < B; ++b) {
        for (int i = 0; i < P->n; ++i) lab[i] = labels[(size_t)i * B + b];
        out[b] = kcut_objective(P, lab);
    }
    free(lab);
    return 0;
}

int kcut_run(const kcut_problem* P, int32_t B, const real* Z0, const real* Y0, const kcut_params* hp,
             uint8_t* labels, double* obj, int32_t* best_restart, real* Zf, real* Yf, real* Xf, int32_t nthreads) {
    const int n = P->n, k = P->k;
    int fail = 0;
    double* best = (double*)malloc(sizeof(double) * (B > 0 ? B : 1));
    if (!best) return 1;
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
#endif
    for (int b = 0; b < B; ++b) {
        const size_t kn = (size_t)k * n;
        real* z = (real*)malloc(sizeof(real) * kn);
        real* zn = (real*)malloc(sizeof(real) * kn);
        real* x = (real*)malloc(sizeof(real) * kn);
        real* y = (real*)malloc(sizeof(real) * n);
        real* yn = (real*)malloc(sizeof(real) * n);
        real* D = (real*)malloc(sizeof(real) * k);
        uint8_t* lab = (uint8_t*)malloc(n);
        uint8_t* bl = (uint8_t*)calloc(n, 1);
        if (!z || !zn || !x || !y || !yn || !D || !lab || !bl) { fail = 1; }
        else {
            double bv = INFINITY;
            for (size_t e = 0; e < kn; ++e) z[e] = Z0[e * B + b];
            for (int i = 0; i < n; ++i) y[i] = Y0[(size_t)i * B + b];
            softmax_cols(n, k, z, x);
            const int T = hp->iters;
            for (int t = 0; t <= T; ++t) {
                const int eval = (t == T) || (t > 0 && t % hp->eval_every == 0);
                if (eval || T == 0) {                            /* label = argmax_j Z_ji, lowest j on ties (K4) */
                    for (int i = 0; i < n; ++i) {
                        int arg = 0;
                        for (int j = 1; j < k; ++j) if (z[(size_t)j * n + i] > z[(size_t)arg * n + i]) arg = j;
                        lab[i] = (uint8_t)arg;
                    }
                    const double v = kcut_objective(P, lab);
                    if (v < bv) { bv = v; memcpy(bl, lab, n); }
                }
                if (t == T) break;
                kcut_step(P, hp, z, x, y, zn, yn, D);
                real* tmp = z; z = zn; zn = tmp;
                tmp = y; y = yn; yn = tmp;
                softmax_cols(n, k, z, x);
            }
            best[b] = bv;
            if (obj) obj[b] = bv;
            if (labels) for (int i = 0; i < n; ++i) labels[(size_t)i * B + b] = bl[i];
            if (Zf) for (size_t e = 0; e < kn; ++e) Zf[e * B + b] = z[e];
            if (Xf) for (size_t e = 0; e < kn; ++e) Xf[e * B + b] = x[e];
            if (Yf) for (int i = 0; i < n; ++i) Yf[(size_t)i * B + b] = y[i];
        }
        free(z); free(zn); free(x); free(y); free(yn); free(D); free(lab); free(bl);
    }
    if (best_restart && !fail) {
        int arg = 0;
        for (int b = 1; b < B; ++b) if (best[b] < best[arg]) arg = b;
        *best_restart = arg;
    }
    free(best);
    return fail;
}
