// gda_internal.cuh -- shared by the translation units of libgda_b200.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/gda.h"

// ---------------------------------------------------------------------------------------------------
// error plumbing
// ---------------------------------------------------------------------------------------------------
void gda_set_error(const char* fmt, ...);

#define GDA_CUDA_TRY(expr)                                                                        \
    do {                                                                                          \
        cudaError_t e__ = (expr);                                                                 \
        if (e__ != cudaSuccess) {                                                                 \
            gda_set_error("%s:%d: %s failed: %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e__)); \
            return GDA_ERR_CUDA;                                                                  \
        }                                                                                         \
    } while (0)

#define GDA_TRY(expr)                        \
    do {                                     \
        gda_status s__ = (expr);             \
        if (s__ != GDA_OK) return s__;       \
    } while (0)

enum { GDA_KIND_SPARSE = 0, GDA_KIND_DENSE = 1, GDA_KIND_MAXSAT = 2, GDA_KIND_KCUT = 3 };

// ---------------------------------------------------------------------------------------------------
// update parameters handed to the kernels by value
// ---------------------------------------------------------------------------------------------------
struct UpdParams {
    float alpha, beta, delta, log_eps;
    uint32_t seed_mix;   // mix32(seed_lo ^ seed_hi * 0x9E3779B9)
    int32_t gfun;
};

// PDBO-s (GDA_DUAL_SCALAR) state handed to the step kernels; mu == nullptr means per-variable duals.
// Sparse path: the step kernel of iteration t reads the multipliers mu^t.  Every block adds the sum of g over the values
// x^{t+1} IT WRITES (fp32, fixed order inside the block) to one of GDA_GACC_WAYS accumulators per restart in 64-bit FIXED
// POINT (2^-32) with integer reductions -- exact, hence independent of the order in which blocks arrive: deterministic.  So
// S^{t+1} = sum_i g(x_i^{t+1}) is complete when the kernel ends, one iteration BEFORE it is needed, and the multiplier update
// mu^{t+1} = mu^t + beta S^t costs no launch of its own: block 0 of every 128-restart chunk of kernel t adds the ways of S^t
// (left by kernel t - 1; by sparse_dual_init for t = 0), writes mu^{t+1} into the other mu buffer and clears them, while the
// rest of the kernel runs (config 3: 22.1 us per iteration with partial rows and a reduce kernel, 19.8 with the fixed-point
// sums and a B-thread finalize kernel, see DESIGN.md for this scheme).  mu and the accumulators follow the parity of x.
// MaxSAT and dense paths: the blocks / epilogue threads leave their sums as rows of gpart and gsum_reduce adds them in a
// fixed order and writes mu^{t+1} (on the MaxSAT kernel the integer reductions measured slower: 52.7 against 46.1 us).
struct ScalarDual {
    const float* mu = nullptr;                 // [B] this step's multipliers mu^t
    unsigned long long* gacc = nullptr;        // [GDA_GACC_WAYS][B] S^t = sum_i g(x_i^t), fixed point (two's complement): complete; consumed and cleared
    unsigned long long* gacc_next = nullptr;   // [GDA_GACC_WAYS][B] S^{t+1}: accumulated by this kernel (zero at its start)
    float* mu_out = nullptr;                   // [B] mu^{t+1}, written by block 0 of every chunk of the launch with advance != 0
    float beta = 0.0f;
    int32_t advance = 0;
    int32_t B = 0;
    float* gpart = nullptr;                    // MaxSAT: [ceil(n / 8)][B]; dense: [n / 128][B]
};
constexpr double GDA_GACC_SCALE = 4294967296.0;   // 2^32
#ifndef GDA_GACC_WAYS_N
#define GDA_GACC_WAYS_N 32
#endif
constexpr int GDA_GACC_WAYS = GDA_GACC_WAYS_N;                 // blocks spread over this many accumulators: few same-address atomics
                                                               // (config 3, us per iteration: 8 ways 19.6, 16 18.3, 32 18.0, 64 18.1, 128 18.2)

// device-side run state (lives in the workspace)
struct RunState {
    uint32_t t;             // iteration index of the iterate currently in x[cur]
    uint32_t n_eval;        // evaluations done so far in this run
    uint32_t ticket;        // blocks of the current finalize launch that are done (reset by the last one)
    uint32_t imp_accum;     // OR of "a restart of my block improved" over the blocks of the current finalize launch
    uint32_t any_improved;  // ... of the last completed evaluation: 0 lets commit_kernel return at once
};

// ---------------------------------------------------------------------------------------------------
// the opaque handle
// ---------------------------------------------------------------------------------------------------
struct Workspace {
    int32_t B = 0;
    int32_t ld = 0;                     // row stride of the state arrays: B, except dense problems (B rounded up to a multiple of 128)
    int32_t parity = 0;                 // which x / zt buffer holds the current iterate
    bool has_state = false;             // a previous gda_run left (x, y, best-so-far) here: x0 == NULL may resume
    float* x[2] = {nullptr, nullptr};   // [n][B] double buffer (Jacobi: every row reads all of x^t)
    float* y = nullptr;                 // [n][B], updated in place
    float* z = nullptr;                 // Max-k-Cut: logits [k][n][B], updated in place (x[] then holds SoftMax(z), [k][n][B])
    uint8_t* lab = nullptr;             // Max-k-Cut: labels of the current iterate at an evaluation, [n][B]
    float* mu[2] = {nullptr, nullptr};  // PDBO-s: [B] multipliers, double-buffered with the parity of x
    float* gpart = nullptr;             // PDBO-s, MaxSAT and dense paths: [n_gpart][B] partial sums of g
    int32_t n_gpart = 0;
    unsigned long long* gacc = nullptr; // PDBO-s, sparse path: [GDA_GACC_WAYS][B] fixed-point sums of g (ScalarDual)
    int32_t dual = 0;                   // dual mode of the state held here
    uint8_t* x_bin = nullptr;           // [n][B] best-so-far rounded point
    double* best_obj = nullptr;         // [B]
    double* obj_now = nullptr;          // [B]
    int32_t* improved = nullptr;        // [B]
    void* partial = nullptr;            // [n_part][B] int64 or double partial objective sums
    int32_t n_part = 0;
    RunState* state = nullptr;
    double* block_min = nullptr;        // [ceil(B / 32)] per-block minima of the best objectives (finalize)
    int32_t* best_restart = nullptr;    // [1]
    double* best_val = nullptr;         // [1]
    double* trace_best = nullptr;       // internal trace buffers (copied out on request)
    uint64_t* trace_ns = nullptr;
    int32_t trace_cap = 0;
    int32_t n_eval_host = 0;            // evaluations recorded in the trace so far (run + resumed runs)
    // dense path
    __nv_bfloat16* zt[2] = {nullptr, nullptr};  // [B][n] bf16 GEMM operand (centred x - 1/2, or x_hat)
    int32_t score_scratch = 1;                  // which zt buffer dense scoring may clobber (the one not holding z^t)
};

struct GraphKey {
    int32_t B = -1, len = 0, parity = 0, with_eval = 0;
    gda_params prm{};
    bool operator==(const GraphKey& o) const;
};
struct CachedGraph {
    GraphKey key;
    cudaGraphExec_t exec = nullptr;
    cudaGraph_t graph = nullptr;
    int64_t launches = 0, step_launches = 0;
};

struct gda_problem {
    int32_t kind = 0;
    int32_t n = 0;
    int32_t n_pad = 0;                   // rows of the state arrays: n, except dense problems (n rounded up to a multiple of 256)
    int64_t nnz = 0;
    int32_t m = 0;
    int32_t kparts = 0;                  // Max-k-Cut: number of parts k (0 otherwise)
    int32_t integral = 0;
    int device = 0;
    int num_sms = 148;
    int64_t l2_bytes = 126 << 20;
    // sparse QUBO: off-diagonal CSR with val2 = Q_ij + Q_ji (= 2 Q_ij), cprime = c + diag(Q)
    int32_t* d_rowptr = nullptr; int32_t* d_col = nullptr; float* d_val2 = nullptr;
    float* d_cprime = nullptr;           // also used by the dense path
    int32_t* d_heavy_rows = nullptr; int32_t n_heavy = 0;   // rows handled by the row-split kernel
    int32_t* d_light_rows = nullptr; int32_t n_light = 0;   // nullptr = all rows, in order
    int32_t* d_local_rows = nullptr;                         // the light rows grouped by adjacency (locality_order), or nullptr
    int32_t max_deg = 0;
    // slab path (small n, gda_sparse.cu): sliced ELL of (column byte offset, val2) pairs, 16 rows per group
    int2* d_slab_ent = nullptr; int32_t* d_slab_goff = nullptr; int32_t* d_slab_grow = nullptr;
    int32_t slab_groups = 0, slab_slots = 0; int64_t slab_real = 0;
    uint16_t* d_slab_ent16 = nullptr; uint32_t slab_cbits = 0; int32_t slab_passes = 0;   // compact form (one |val2|), else null
    int32_t slab_mode = 0;               // GDA_OPT_SPARSE_PATH: 1 "slab" always, -1 "stream" never, 0 by the cost model
    // the other per-handle options of gda_set_option (include/gda.h); a change drops the cached graphs
    int32_t opt_split_all = -1;          // GDA_OPT_SPLIT_ALL_ROWS: -1 by the rule, 0 rows whole, 1 every row through the row-split kernel
    int32_t opt_narrow_split = 1;        // GDA_OPT_NARROW_SPLIT: lane groups share long rows in the narrow sparse step
    int32_t opt_maxsat_narrow = 1;       // GDA_OPT_MAXSAT_NARROW: slot groups in the MaxSAT step for B <= 64
    int32_t opt_dense_shape = -1;        // GDA_OPT_DENSE_SHAPE: -1 the largest cluster shape that pays, 0..3 at most this shape
    int32_t opt_graphs = 1;              // GDA_OPT_GRAPHS: replay captured chunks (1) or enqueue the kernels directly (0)
    int32_t opt_row_grouping = 1;        // GDA_OPT_ROW_GROUPING: PDBO-s sparse step walks the rows grouped by adjacency
    int32_t* d_ell = nullptr;            // [n][16] packed low-degree rows: 8 cols + 8 val2 (see gda_sparse.cu); nullptr = not built
    // dense QUBO: Q_off in bf16 [n][n] (zero diagonal), r0 = Q_off 1 (row sums) for the centred operand
    __nv_bfloat16* d_Qbf = nullptr; float* d_rowsum = nullptr;
    void* tmap_Q = nullptr;              // CUtensorMap (128 B), host copy
    // MaxSAT: per occurrence slot (variable-major): coef = w_j * s_ji, others[kw] signed literals (0 = pad)
    int32_t* d_vptr = nullptr; float* d_coef = nullptr; int32_t* d_others = nullptr; int32_t kw = 0;
    int32_t* d_cptr = nullptr; int32_t* d_lit = nullptr; float* d_w = nullptr; int32_t kmax = 0, kmin = 0;
    Workspace ws;
    cudaStream_t own_stream = nullptr;   // used when the caller passes the legacy default stream (not capturable)
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaEvent_t ev_last = nullptr;       // recorded after everything an entry point enqueued (what destroy / reallocation wait for)
    std::vector<CachedGraph> graphs;
    int64_t last_launches = 0, last_step_launches = 0;
};

// ---------------------------------------------------------------------------------------------------
// kernels' launchers, one translation unit per path.  Every launcher enqueues on `s` and returns the
// number of kernels it launched through *launches (may be nullptr).
// ---------------------------------------------------------------------------------------------------
// sparse QUBO (gda_sparse.cu)
gda_status sparse_step(gda_problem* p, int32_t B, const float* x, float* y, float* xn, const UpdParams& up,
                       const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s, int64_t* launches);
gda_status sparse_configure(gda_problem* p);                       // at create
// small n: sliced-ELL structure built at create, and one launch per chunk (steps + evaluation) when it applies
gda_status sparse_build_slab(gda_problem* p, const std::vector<int32_t>& rowptr, const std::vector<int32_t>& col,
                             const std::vector<float>& val2);
gda_status sparse_chunk_slab(gda_problem* p, int32_t B_eval, int32_t B, int32_t len, const float* x_in, float* x_out, float* y,
                             const float* mu_in, float* mu_out,     // PDBO-s: [B] multipliers before / after the chunk; NULL = PDBO
                             const UpdParams& up, cudaStream_t s, int64_t* launches, int* done);
gda_status sparse_grad(gda_problem* p, int32_t B, const float* x, float* G, cudaStream_t s);
gda_status sparse_score_partials(gda_problem* p, int32_t B, const float* x, void* partial, int32_t* n_part,
                                 cudaStream_t s, int64_t* launches);
int32_t sparse_num_partials(const gda_problem* p, int32_t B);
// f(x) (continuous x) as per-block partial sums, one row per block of 64 rows; returns the rows written
gda_status sparse_value_partials(gda_problem* p, int32_t B, const float* x, double* partial, int32_t* n_part, cudaStream_t s);

// MaxSAT (gda_maxsat.cu)
gda_status maxsat_step(gda_problem* p, int32_t B, const float* x, float* y, float* xn, const UpdParams& up,
                       const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s, int64_t* launches);
int32_t maxsat_num_gparts(const gda_problem* p);
gda_status maxsat_grad(gda_problem* p, int32_t B, const float* x, float* G, cudaStream_t s);
gda_status maxsat_score_partials(gda_problem* p, int32_t B, const float* x, void* partial, int32_t* n_part,
                                 cudaStream_t s, int64_t* launches);
int32_t maxsat_num_partials(const gda_problem* p, int32_t B);
gda_status maxsat_value_partials(gda_problem* p, int32_t B, const float* x, double* partial, int32_t* n_part, cudaStream_t s);

// Max-k-Cut (gda_kcut.cu): x = SoftMax(z) planes [k][n][B]
gda_status kcut_step(gda_problem* p, int32_t B, const float* x, float* z, float* y, float* xn, const UpdParams& up,
                     cudaStream_t s, int64_t* launches);
gda_status kcut_softmax(gda_problem* p, int32_t B, const float* z, float* x, cudaStream_t s, int64_t* launches);
gda_status kcut_score_partials(gda_problem* p, int32_t B, const float* z, uint8_t* lab, void* partial, int32_t* n_part,
                               cudaStream_t s, int64_t* launches);
gda_status kcut_grad(gda_problem* p, int32_t B, const float* x, float* G, cudaStream_t s);                 // x = SoftMax(z), [k][n][B]
gda_status kcut_value_partials(gda_problem* p, int32_t B, const float* x, const float* y, float y_scalar, int32_t gfun,
                               double* partial, int32_t* n_part, cudaStream_t s);
gda_status kcut_commit(gda_problem* p, int32_t B, const uint8_t* lab, const int32_t* improved, uint8_t* x_bin,
                       cudaStream_t s, int64_t* launches);
int32_t kcut_num_partials(const gda_problem* p, int32_t B);

// dense QUBO (gda_dense.cu)
gda_status dense_prepare(gda_problem* p, const float* Q_host, const float* c_host);   // at create
gda_status dense_make_operand(gda_problem* p, int32_t B, const float* x, __nv_bfloat16* zt, int hat,
                              cudaStream_t s, int64_t* launches);
gda_status dense_step(gda_problem* p, int32_t B, float* x, float* y, const __nv_bfloat16* zt_in,
                      __nv_bfloat16* zt_out, const UpdParams& up, const ScalarDual& sd, const RunState* st, uint32_t t_off,
                      cudaStream_t s, int64_t* launches);
gda_status dense_grad(gda_problem* p, int32_t B, const float* x, float* G, cudaStream_t s);
gda_status dense_score_partials(gda_problem* p, int32_t B, const float* x, void* partial, int32_t* n_part,
                                cudaStream_t s, int64_t* launches);
int32_t dense_num_partials(const gda_problem* p, int32_t B);
void dense_release(gda_problem* p);

// shared evaluation tail (gda_eval.cu)
gda_status eval_finalize(gda_problem* p, int32_t B, int32_t ld, const void* partial, int32_t n_part, double* obj_now,
                         double* best_obj, int32_t* improved, RunState* st, double* trace_best,
                         uint64_t* trace_ns, int32_t trace_cap, uint32_t advance_t, cudaStream_t s,
                         int64_t* launches);
gda_status eval_commit(gda_problem* p, int32_t ld, const float* x, const int32_t* improved, uint8_t* x_bin,
                       cudaStream_t s, int64_t* launches);
gda_status eval_argbest(int32_t B, const double* obj, int32_t* best_restart, double* best_val,
                        cudaStream_t s, int64_t* launches);
// sum_i y_i g(x_i) as partial sums over blocks of 64 rows (y == nullptr: y_scalar); double reduction of partial rows
gda_status eval_yg_partials(gda_problem* p, int32_t n_rows, int32_t B, const float* x, const float* y, float y_scalar, int32_t gfun,
                            float log_eps, double* partial, int32_t* n_part, cudaStream_t s);
gda_status eval_sum_partials(int32_t B, int32_t ld, const double* partial, int32_t n_part, double* out, cudaStream_t s);
// dense Lagrangian: partial[rb][b] = sum over the 64 rows of block rb of x_i (G_i + c'_i) / 2  (= f(x) with G = grad f)
gda_status eval_xg_partials(gda_problem* p, int32_t ld, const float* x, const float* G, double* partial, int32_t* n_part, cudaStream_t s);
gda_status eval_count_ones(gda_problem* p, int32_t B, const uint8_t* x_bin, int32_t* ones, cudaStream_t s, int64_t* launches);
gda_status run_init(gda_problem* p, int32_t B, const float* x0, const float* l0, float l0_scalar,
                    uint32_t t0, cudaStream_t s, int64_t* launches);
gda_status score_reduce(gda_problem* p, int32_t B, int32_t ld, const void* partial, int32_t n_part, double* obj,
                        cudaStream_t s);
// PDBO-s: mu_out[b] = mu_in[b] + beta * sum_r gpart[r][b], summed in a fixed order (deterministic)
gda_status gsum_reduce(int32_t B, const float* gpart, int32_t n_gpart, float beta, const float* mu_in, float* mu_out,
                       cudaStream_t s, int64_t* launches);
gda_status mu_init(int32_t B, const float* l0, float l0_scalar, float* mu, cudaStream_t s, int64_t* launches);
// PDBO-s, sparse / MaxSAT: mu_out[b] = mu_in[b] + beta * (sum of the ways of gacc[.][b]) / 2^32; clears gacc
gda_status sparse_dual_init(gda_problem* p, int32_t B, const float* x, int32_t gfun, float log_eps, unsigned long long* gacc, cudaStream_t s,
                            int64_t* launches);      // S^0 = sum_i g(x_i^0) into the accumulators (start of a PDBO-s run)

// ---------------------------------------------------------------------------------------------------
// device helpers: g, g', the fused update S4 (Eq. 6 + perturbation), the tie-break hash
// ---------------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__host__ __device__ __forceinline__ uint32_t mix32(uint32_t h) {
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    return h;
}

// s = +1 / -1 from (seed, t, i, b): DESIGN.md reading R3 (the oracle writes the same integer function out itself)
__device__ __forceinline__ float side_from_hash(uint32_t seed_mix, uint32_t t, uint32_t i, uint32_t b) {
    uint32_t h = mix32(seed_mix + t);
    h = mix32(h + i);
    h = mix32(h + b);
    return (h & 1u) ? 1.0f : -1.0f;
}

// natural log through MUFU.LG2 (__logf: abs error <= 2^-21.4 on [0.5, 2], <= 3 ulp elsewhere): with alpha*y and beta
// of order 1e-2 that is < 1e-7 on x+ and y+, two orders below the 1e-5 step tolerance
__device__ __forceinline__ float fast_ln(float u) { return __logf(u); }

// One element of S4: (x, y, G) at time t -> (x, y) at time t+1.   PAPER.md:136-142 (Eq. 6), 148, 732.
// Split in two so that vector callers can test the (rare) perturbation condition once for several elements:
// gda_update_nopert is Eq. 6 alone; gda_perturb applies reading R3/R3a to the tentative point.
template <int GFUN>
__device__ __forceinline__ void gda_update_nopert(float x, float y, float G, const UpdParams& up, float& xt, float& yn) {
    float gp, gv;
    if (GFUN == GDA_G_QUADRATIC) {
        gp = 2.0f * x - 1.0f;
        gv = x * x - x;
    } else {
        // Reading R4: g'(x) = ln(xc) - ln(1 - xc), xc = clip(x, eps, 1 - eps); g(x) = x ln x + (1-x) ln(1-x), 0 at the ends.
        // Evaluated branch-free from two logs of a = max(x, eps), b = max(1 - x, eps) (1 - x is exact in fp32 near 1,
        // whereas 1 - eps is not representable):
        //   g' = ln a - ln b        differs from the clipped form only for x outside [eps, 1-eps], by <= eps = 1e-6
        //   g  = x ln a + (1-x) ln b   exact 0 at x = 0 and 1; for 0 < x < eps it is x ln eps instead of x ln x,
        //                              an absolute difference <= eps/e = 3.7e-7
        // i.e. <= alpha*y*1e-6 on x+ and <= beta*3.7e-7 on y+, far below the 1e-5 step tolerance.
        const float u = 1.0f - x;
        const float l0 = fast_ln(fmaxf(x, up.log_eps)), l1 = fast_ln(fmaxf(u, up.log_eps));
        gp = l0 - l1;
        gv = fmaf(x, l0, u * l1);
    }
    xt = x - up.alpha * (G + y * gp);
    xt = fminf(fmaxf(xt, 0.0f), 1.0f);
    yn = y + up.beta * gv;
}

// g(x) alone (PDBO-s sums it over the variables of a restart); same expressions as in gda_update_nopert
template <int GFUN>
__device__ __forceinline__ float gda_g(float x, const UpdParams& up) {
    if (GFUN == GDA_G_QUADRATIC) return x * x - x;
    const float u = 1.0f - x;
    return fmaf(x, fast_ln(fmaxf(x, up.log_eps)), u * fast_ln(fmaxf(u, up.log_eps)));
}

__device__ __forceinline__ bool gda_in_band(float x, float xt, float delta) {
    return fabsf(x - 0.5f) < delta && fabsf(xt - 0.5f) < delta;           // false for delta == 0
}

__device__ __forceinline__ float gda_perturb(float x, float xt, float delta, uint32_t seed_mix, uint32_t t, uint32_t i, uint32_t b) {
    float s;
    if (xt > 0.5f) s = 1.0f; else if (xt < 0.5f) s = -1.0f;
    else if (x > 0.5f) s = 1.0f; else if (x < 0.5f) s = -1.0f;
    else s = side_from_hash(seed_mix, t, i, b);
    xt = 0.5f + delta * s;
    if (fabsf(xt - 0.5f) < delta)                              // rounding fell inside: one ulp away from 1/2
        xt = __int_as_float(__float_as_int(xt) + (s > 0.0f ? 1 : -1));
    return xt;
}

template <int GFUN>
__device__ __forceinline__ void gda_update(float x, float y, float G, const UpdParams& up, uint32_t t,
                                           uint32_t i, uint32_t b, float& xn, float& yn) {
    float xt;
    gda_update_nopert<GFUN>(x, y, G, up, xt, yn);
    if (gda_in_band(x, xt, up.delta)) xt = gda_perturb(x, xt, up.delta, up.seed_mix, t, i, b);
    xn = xt;
}

// Four consecutive restarts b0..b0+3 of variable i: one test for the rare perturbation branch.
template <int GFUN>
__device__ __forceinline__ void gda_update4(const float4& x, const float4& y, const float4& G, const UpdParams& up,
                                            uint32_t t, uint32_t i, uint32_t b0, float4& xn, float4& yn) {
    gda_update_nopert<GFUN>(x.x, y.x, G.x, up, xn.x, yn.x);
    gda_update_nopert<GFUN>(x.y, y.y, G.y, up, xn.y, yn.y);
    gda_update_nopert<GFUN>(x.z, y.z, G.z, up, xn.z, yn.z);
    gda_update_nopert<GFUN>(x.w, y.w, G.w, up, xn.w, yn.w);
    const bool b_x = gda_in_band(x.x, xn.x, up.delta), b_y = gda_in_band(x.y, xn.y, up.delta);
    const bool b_z = gda_in_band(x.z, xn.z, up.delta), b_w = gda_in_band(x.w, xn.w, up.delta);
    if (b_x | b_y | b_z | b_w) {
        if (b_x) xn.x = gda_perturb(x.x, xn.x, up.delta, up.seed_mix, t, i, b0 + 0);
        if (b_y) xn.y = gda_perturb(x.y, xn.y, up.delta, up.seed_mix, t, i, b0 + 1);
        if (b_z) xn.z = gda_perturb(x.z, xn.z, up.delta, up.seed_mix, t, i, b0 + 2);
        if (b_w) xn.w = gda_perturb(x.w, xn.w, up.delta, up.seed_mix, t, i, b0 + 3);
    }
}


__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

// ---- PDBO-s helpers shared by the warp-per-(row, chunk) step kernels -------------------------------------------
// scalar_dual_commit: ONE warp adds its block's sums t (lane = float4 of restarts c4) to accumulator `way`.
__device__ __forceinline__ void scalar_dual_commit(float4 t, bool active, int c4, unsigned way, const ScalarDual& sd) {
    if (!active) return;
    unsigned long long* acc = sd.gacc_next + (size_t)(way % GDA_GACC_WAYS) * sd.B + 4 * c4;
    atomicAdd(acc + 0, (unsigned long long)__double2ll_rn((double)t.x * GDA_GACC_SCALE));
    atomicAdd(acc + 1, (unsigned long long)__double2ll_rn((double)t.y * GDA_GACC_SCALE));
    atomicAdd(acc + 2, (unsigned long long)__double2ll_rn((double)t.z * GDA_GACC_SCALE));
    atomicAdd(acc + 3, (unsigned long long)__double2ll_rn((double)t.w * GDA_GACC_SCALE));
}

// A block of NW warps closes the multiplier update for the 128 restarts of its chunk (lane = float4 of restarts c4):
// mu^{t+1} = mu^t + beta S^t, S^t the exact integer sum of the ways, and clears the ways.  Warp w takes the ways
// w, w + NW, ... (four independent 16-byte loads per lane and way: one round trip), warp 0 adds the warps' sums.
// Must be called by every thread of the block.
template <int NW>
__device__ __forceinline__ void scalar_dual_advance(long long (*adv)[32][4], int warp, int lane, bool active, int c4,
                                                    const ScalarDual& sd) {
    long long t[4] = {0, 0, 0, 0};
    if (active) {
        for (int k = warp; k < GDA_GACC_WAYS; k += NW) {
            ulonglong2* p = reinterpret_cast<ulonglong2*>(sd.gacc + (size_t)k * sd.B + 4 * c4);
            const ulonglong2 a = p[0], b = p[1];
            t[0] += (long long)a.x; t[1] += (long long)a.y; t[2] += (long long)b.x; t[3] += (long long)b.y;
            p[0] = make_ulonglong2(0ull, 0ull); p[1] = make_ulonglong2(0ull, 0ull);
        }
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) adv[warp][lane][q] = t[q];
    __syncthreads();
    if (warp != 0 || !active) return;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        long long s = adv[0][lane][q];
        for (int w = 1; w < NW; ++w) s += adv[w][lane][q];
        const int b = 4 * c4 + q;
        sd.mu_out[b] = sd.mu[b] + sd.beta * (float)((double)s / GDA_GACC_SCALE);
    }
}

// Called by every thread of a block whose NW warps hold their sums of g in gs (0 for warps / lanes without work): the
// warps' sums are added in warp order by warp 0, which then commits them.
// One gpart row per block (MaxSAT path): the NW warps' sums of g, added in warp order by warp 0; gsum_reduce adds the rows.
template <int NW>
__device__ __forceinline__ void scalar_dual_block_sum(float4 gs, float4 (*red)[32], int warp, int lane, bool active,
                                                      float* __restrict__ gpart_row_c4) {
    red[warp][lane] = gs;
    __syncthreads();
    if (warp != 0 || !active) return;
    float4 t = red[0][lane];
#pragma unroll
    for (int w = 1; w < NW; ++w) { const float4 r = red[w][lane]; t.x += r.x; t.y += r.y; t.z += r.z; t.w += r.w; }
    *reinterpret_cast<float4*>(gpart_row_c4) = t;
}

template <int NW>
__device__ __forceinline__ void scalar_dual_finish(float4 gs, float4 (*red)[32], int warp, int lane, bool active, int c4,
                                                   unsigned way, const ScalarDual& sd) {
    red[warp][lane] = gs;
    __syncthreads();
    if (warp != 0) return;
    float4 t = red[0][lane];
#pragma unroll
    for (int w = 1; w < NW; ++w) { const float4 r = red[w][lane]; t.x += r.x; t.y += r.y; t.z += r.z; t.w += r.w; }
    scalar_dual_commit(t, active, c4, way, sd);
}

#endif
