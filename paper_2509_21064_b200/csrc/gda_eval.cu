// gda_eval.cu -- the evaluation tail shared by all three problem kinds (S5 bookkeeping, S6 arg-best):
//   fixed-order reduction of the per-block partial objective sums, best-so-far per restart
//   ("retaining the best solution"; reading R5), committing x_hat of improved restarts,
//   the best-vs-time trace and the final argmin over restarts (reading R6).
#include "gda_internal.cuh"

#include <math_constants.h>
#include <algorithm>

namespace {

constexpr int FIN_COLS = 32, FIN_SLICES = 32;                // block = 32 restarts x 32 row slices

__device__ __forceinline__ uint64_t globaltimer_ns() {
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// obj_now[b] = sum_p partial[p][b]; best-so-far update.  grid = ceil(B / 32) blocks of (32 restarts, 32 row slices):
// slice s adds the rows p = s, s + 32, ... (8 independent loads in flight), the 32 slice sums are then added in slice
// order -- a fixed order, so the result is deterministic (and exact for integral instances).  The last block to finish
// (a ticket in the run state) takes the minimum of the blocks' best values -- order-independent -- records the trace
// entry, advances the run state and publishes whether ANY restart improved, which lets the commit kernel return at once.
// ld = row stride of `partial` (>= B).
template <bool INTEGRAL>
__global__ void __launch_bounds__(FIN_COLS * FIN_SLICES)
finalize_kernel(int B, int ld, const void* __restrict__ partial, int n_part, double* __restrict__ obj_now,
                double* __restrict__ best_obj, int32_t* __restrict__ improved, RunState* st, double* block_min,
                double* __restrict__ trace_best, uint64_t* __restrict__ trace_ns, int trace_cap, uint32_t advance_t) {
    using acc_t = typename std::conditional<INTEGRAL, long long, double>::type;
    __shared__ acc_t red[FIN_SLICES][FIN_COLS + 1];
    const acc_t* part = reinterpret_cast<const acc_t*>(partial);
    const int col = threadIdx.x, slice = threadIdx.y;
    const int b = blockIdx.x * FIN_COLS + col;
    acc_t s = 0;
    if (b < B) {
        int q = slice;
        for (; q + 7 * FIN_SLICES < n_part; q += 8 * FIN_SLICES) {
            acc_t v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = part[(size_t)(q + u * FIN_SLICES) * ld + b];
#pragma unroll
            for (int u = 0; u < 8; ++u) s += v[u];
        }
        for (; q < n_part; q += FIN_SLICES) s += part[(size_t)q * ld + b];
    }
    red[slice][col] = s;
    __syncthreads();
    if (slice != 0) return;                                  // warp 0 = the 32 restarts of this block
    double local_min = CUDART_INF;
    int imp = 0;
    if (b < B) {
        acc_t t = red[0][col];
#pragma unroll
        for (int k = 1; k < FIN_SLICES; ++k) t += red[k][col];
        const double v = (double)t;
        if (obj_now) obj_now[b] = v;
        if (best_obj) {
            double best = best_obj[b];
            imp = v < best;
            if (imp) { best = v; best_obj[b] = v; }
            improved[b] = imp;
            local_min = best;
        }
    }
    if (!st) return;
    for (int o = 16; o > 0; o >>= 1) local_min = fmin(local_min, __shfl_xor_sync(0xffffffffu, local_min, o));
    imp = __any_sync(0xffffffffu, imp);
    unsigned ticket = 0;
    if (col == 0) {
        block_min[blockIdx.x] = local_min;
        if (imp) atomicOr(&st->imp_accum, 1u);
        __threadfence();
        ticket = atomicAdd(&st->ticket, 1u);
    }
    ticket = __shfl_sync(0xffffffffu, ticket, 0);
    if (ticket != gridDim.x - 1) return;
    __threadfence();                                         // last block: every block's minimum is visible
    double m = CUDART_INF;
    for (int k = col; k < (int)gridDim.x; k += 32) m = fmin(m, __ldcg(block_min + k));
    for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (col == 0) {
        const uint32_t k = st->n_eval;
        if (trace_best && (int)k < trace_cap) { trace_best[k] = m; trace_ns[k] = globaltimer_ns(); }
        st->n_eval = k + 1;
        st->t += advance_t;
        st->any_improved = atomicExch(&st->imp_accum, 0u);
        st->ticket = 0;
    }
}

// x_bin[:, b] = [x[:, b] > 1/2] for every restart b whose objective improved at this evaluation; returns at once when
// none did (the usual case late in a run).  Grid-stride over float4 vectors.
__global__ void __launch_bounds__(256)
commit_kernel(size_t n_vec, int B4, const float* __restrict__ x, const int32_t* __restrict__ improved,
              const RunState* __restrict__ st, uint8_t* __restrict__ x_bin) {
    if (st && st->any_improved == 0u) return;
    for (size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x; v < n_vec; v += (size_t)gridDim.x * blockDim.x) {
        const int c4 = (int)(v % (size_t)B4);
        const int4 imp = __ldg(reinterpret_cast<const int4*>(improved) + c4);
        if (!(imp.x | imp.y | imp.z | imp.w)) continue;
        const float4 xv = ldg4(x + 4 * v);
        uchar4 o = reinterpret_cast<uchar4*>(x_bin)[v];
        if (imp.x) o.x = xv.x > 0.5f;
        if (imp.y) o.y = xv.y > 0.5f;
        if (imp.z) o.z = xv.z > 0.5f;
        if (imp.w) o.w = xv.w > 0.5f;
        reinterpret_cast<uchar4*>(x_bin)[v] = o;
    }
}

// S6: argmin over restarts, ties -> lowest index; warp shuffles, then one warp over the per-warp winners
__global__ void __launch_bounds__(256)
argbest_kernel(int B, const double* __restrict__ obj, int32_t* __restrict__ best_restart,
               double* __restrict__ best_val) {
    __shared__ double sv[8];
    __shared__ int si[8];
    double v = CUDART_INF;
    int idx = 0x7fffffff;
    for (int b = threadIdx.x; b < B; b += blockDim.x) {
        const double o = obj[b];
        if (o < v || (o == v && b < idx)) { v = o; idx = b; }
    }
    for (int off = 16; off > 0; off >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, v, off);
        const int oi = __shfl_xor_sync(0xffffffffu, idx, off);
        if (ov < v || (ov == v && oi < idx)) { v = ov; idx = oi; }
    }
    if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = v; si[threadIdx.x >> 5] = idx; }
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < 8 ? sv[threadIdx.x] : CUDART_INF;
        idx = threadIdx.x < 8 ? si[threadIdx.x] : 0x7fffffff;
        for (int off = 4; off > 0; off >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, v, off);
            const int oi = __shfl_xor_sync(0xffffffffu, idx, off);
            if (ov < v || (ov == v && oi < idx)) { v = ov; idx = oi; }
        }
        if (threadIdx.x == 0) {
            *best_restart = (idx == 0x7fffffff) ? 0 : idx;      // all +inf / NaN: restart 0
            if (best_val) *best_val = (idx == 0x7fffffff) ? obj[0] : v;
        }
    }
}

__global__ void __launch_bounds__(256)
fill_kernel(size_t n_vec, float4* __restrict__ dst, float v) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_vec) dst[i] = make_float4(v, v, v, v);
}

__global__ void __launch_bounds__(256)
init_state_kernel(int B, double* __restrict__ best_obj, int32_t* __restrict__ improved, RunState* st, uint32_t t0) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < B) { best_obj[b] = CUDART_INF; improved[b] = 0; }
    if (b == 0) { st->t = t0; st->n_eval = 0; st->ticket = 0; st->imp_accum = 0; st->any_improved = 1; }
}

// PDBO-s: mu_out[b] = mu_in[b] + beta * sum_r gpart[r][b].  grid ceil(B/32), block (32 restarts, 32 slices): rows are
// dealt to the slices (8 independent loads in flight per thread), every slice and then the slices are added in index
// order, so the sum is deterministic.  (A version with 64 row groups per column block and a last-block-done second
// stage -- threadfence + counter -- was slower: 13 us against 5 us under ncu.)
__global__ void __launch_bounds__(1024)
gsum_reduce_kernel(int B, const float* __restrict__ gpart, int n_gpart, float beta, const float* __restrict__ mu_in,
                   float* __restrict__ mu_out) {
    __shared__ float red[32][33];
    const int tx = threadIdx.x, slice = threadIdx.y;
    const int b = blockIdx.x * 32 + tx;
    float acc = 0.0f;
    if (b < B) {
        int r = slice;
        for (; r + 7 * 32 < n_gpart; r += 8 * 32) {
            float v[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) v[q] = __ldg(gpart + (size_t)(r + 32 * q) * B + b);
#pragma unroll
            for (int q = 0; q < 8; ++q) acc += v[q];
        }
        for (; r < n_gpart; r += 32) acc += __ldg(gpart + (size_t)r * B + b);
    }
    red[slice][tx] = acc;
    __syncthreads();
    if (slice == 0 && b < B) {
        float t = 0.0f;
#pragma unroll
        for (int k = 0; k < 32; ++k) t += red[k][tx];
        mu_out[b] = mu_in[b] + beta * t;
    }
}

// partial[rb][b] = sum over the 64 rows of block rb of y_i g(x_i)   (the constraint part of L)
template <int GFUN>
__global__ void __launch_bounds__(256)
yg_partials_kernel(int n, int B, const float* __restrict__ x, const float* __restrict__ y, float y_scalar,
                   UpdParams up, double* __restrict__ partial) {
    __shared__ double red[8][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c4 = blockIdx.y * 32 + lane;
    const bool active = 4 * c4 < B;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    if (active)
        for (int r = warp; r < 64; r += 8) {
            const int row = blockIdx.x * 64 + r;
            if (row >= n) break;
            const size_t off = (size_t)row * B + 4 * c4;
            const float4 xv = ldg4(x + off);
            const float4 yv = y ? ldg4(y + off) : make_float4(y_scalar, y_scalar, y_scalar, y_scalar);
            acc[0] += (double)(yv.x * gda_g<GFUN>(xv.x, up)); acc[1] += (double)(yv.y * gda_g<GFUN>(xv.y, up));
            acc[2] += (double)(yv.z * gda_g<GFUN>(xv.z, up)); acc[3] += (double)(yv.w * gda_g<GFUN>(xv.w, up));
        }
#pragma unroll
    for (int q = 0; q < 4; ++q) red[warp][lane][q] = acc[q];
    __syncthreads();
    if (warp == 0 && active)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            double t = red[0][lane][q];
            for (int w = 1; w < 8; ++w) t += red[w][lane][q];
            partial[(size_t)blockIdx.x * B + 4 * c4 + q] = t;
        }
}

// dense f(x) at a continuous point from its gradient: f = sum_i x_i ((Q_off x)_i + c'_i) and G = 2 Q_off x + c', so
// f = sum_i x_i (G_i + c'_i) / 2.  partial[rb][b] over blocks of 64 rows; products in fp32, sums in fp64.
__global__ void __launch_bounds__(256)
xg_partials_kernel(int n, int B, const float* __restrict__ x, const float* __restrict__ G, const float* __restrict__ cprime,
                   double* __restrict__ partial) {
    __shared__ double red[8][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c4 = blockIdx.y * 32 + lane;
    const bool active = 4 * c4 < B;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    if (active)
        for (int r = warp; r < 64; r += 8) {
            const int row = blockIdx.x * 64 + r;
            if (row >= n) break;
            const size_t off = (size_t)row * B + 4 * c4;
            const float4 xv = ldg4(x + off), gv = ldg4(G + off);
            const float cp = __ldg(cprime + row);
            acc[0] += (double)(0.5f * xv.x * (gv.x + cp)); acc[1] += (double)(0.5f * xv.y * (gv.y + cp));
            acc[2] += (double)(0.5f * xv.z * (gv.z + cp)); acc[3] += (double)(0.5f * xv.w * (gv.w + cp));
        }
#pragma unroll
    for (int q = 0; q < 4; ++q) red[warp][lane][q] = acc[q];
    __syncthreads();
    if (warp == 0 && active)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            double t = red[0][lane][q];
            for (int w = 1; w < 8; ++w) t += red[w][lane][q];
            partial[(size_t)blockIdx.x * B + 4 * c4 + q] = t;
        }
}

// ones[b] = sum_i x_bin[i][b]: block = 128 restarts (uchar4 per lane) x 32 row slices, integer sums
__global__ void __launch_bounds__(1024)
count_ones_kernel(int n, int B, int ld, const uint8_t* __restrict__ x_bin, int32_t* __restrict__ ones) {
    __shared__ int red[32][32][4];
    const int lane = threadIdx.x, slice = threadIdx.y;
    const int c = blockIdx.x * 128 + 4 * lane;
    int acc[4] = {0, 0, 0, 0};
    if (c < B)
        for (int i = slice; i < n; i += 32) {
            const uchar4 v = *reinterpret_cast<const uchar4*>(x_bin + (size_t)i * ld + c);
            acc[0] += v.x; acc[1] += v.y; acc[2] += v.z; acc[3] += v.w;
        }
#pragma unroll
    for (int q = 0; q < 4; ++q) red[slice][lane][q] = acc[q];
    __syncthreads();
    if (slice == 0 && c < B)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            int t = 0;
            for (int k = 0; k < 32; ++k) t += red[k][lane][q];
            if (c + q < B) ones[c + q] = t;                  // the caller's buffer is [B]: padding restarts are not stored
        }
}

__global__ void mu_init_kernel(int B, const float* __restrict__ l0, float l0_scalar, float* __restrict__ mu) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < B) mu[b] = l0 ? l0[b] : l0_scalar;
}

}  // namespace

gda_status gsum_reduce(int32_t B, const float* gpart, int32_t n_gpart, float beta, const float* mu_in, float* mu_out,
                       cudaStream_t s, int64_t* launches) {
    gsum_reduce_kernel<<<(unsigned)((B + 31) / 32), dim3(32, 32), 0, s>>>(B, gpart, n_gpart, beta, mu_in, mu_out);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status mu_init(int32_t B, const float* l0, float l0_scalar, float* mu, cudaStream_t s, int64_t* launches) {
    mu_init_kernel<<<(B + 255) / 256, 256, 0, s>>>(B, l0, l0_scalar, mu);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

// [rows][B] at the caller (host or device: cudaMemcpyDefault tells by unified addressing) -> [..][ld] in the workspace
static gda_status copy_in(void* dst, size_t ld, const void* src, size_t B, size_t rows, size_t esz, cudaStream_t s) {
    if (ld == B) GDA_CUDA_TRY(cudaMemcpyAsync(dst, src, rows * B * esz, cudaMemcpyDefault, s));
    else GDA_CUDA_TRY(cudaMemcpy2DAsync(dst, ld * esz, src, B * esz, B * esz, rows, cudaMemcpyDefault, s));
    return GDA_OK;
}

gda_status run_init(gda_problem* p, int32_t B, const float* x0, const float* l0, float l0_scalar,
                    uint32_t t0, cudaStream_t s, int64_t* launches) {
    Workspace& ws = p->ws;
    const size_t ld = (size_t)ws.ld, elems = (size_t)p->n_pad * ld;          // padding: restarts up to a multiple of 4 (dense: 128), dense variables up to 256
    const bool padded = ld != (size_t)B || p->n_pad != p->n;
    if (p->kind == GDA_KIND_KCUT) {
        if (padded) GDA_CUDA_TRY(cudaMemsetAsync(ws.z, 0, elems * p->kparts * sizeof(float), s));   // padding restarts: logits 0
        GDA_TRY(copy_in(ws.z, ld, x0, (size_t)B, (size_t)p->n * p->kparts, sizeof(float), s));
    } else {
        if (padded) GDA_CUDA_TRY(cudaMemsetAsync(ws.x[0], 0, elems * sizeof(float), s));   // padding variables and restarts start at 0
        GDA_TRY(copy_in(ws.x[0], ld, x0, (size_t)B, (size_t)p->n, sizeof(float), s));
    }
    if (ws.dual == GDA_DUAL_SCALAR) {
        if (ws.gacc)                                         // nothing pending from an earlier (possibly failed) run; both parities
            GDA_CUDA_TRY(cudaMemsetAsync(ws.gacc, 0, 2 * (size_t)GDA_GACC_WAYS * ld * sizeof(unsigned long long), s));
        GDA_TRY(mu_init((int32_t)ld, nullptr, l0 ? 0.0f : l0_scalar, ws.mu[0], s, launches));
        if (l0) GDA_CUDA_TRY(cudaMemcpyAsync(ws.mu[0], l0, (size_t)B * sizeof(float), cudaMemcpyDefault, s));
    } else if (l0) {
        if (padded) GDA_CUDA_TRY(cudaMemsetAsync(ws.y, 0, elems * sizeof(float), s));
        GDA_TRY(copy_in(ws.y, ld, l0, (size_t)B, (size_t)p->n, sizeof(float), s));
    } else {
        const size_t n_vec = elems / 4;
        fill_kernel<<<(unsigned)((n_vec + 255) / 256), 256, 0, s>>>(n_vec, reinterpret_cast<float4*>(ws.y), l0_scalar);
        if (launches) ++*launches;
    }
    GDA_CUDA_TRY(cudaMemsetAsync(ws.x_bin, 0, elems, s));
    init_state_kernel<<<(unsigned)((ld + 255) / 256), 256, 0, s>>>((int)ld, ws.best_obj, ws.improved, ws.state, t0);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status eval_finalize(gda_problem* p, int32_t B, int32_t ld, const void* partial, int32_t n_part, double* obj_now,
                         double* best_obj, int32_t* improved, RunState* st, double* trace_best,
                         uint64_t* trace_ns, int32_t trace_cap, uint32_t advance_t, cudaStream_t s,
                         int64_t* launches) {
    const unsigned grid = (unsigned)((B + FIN_COLS - 1) / FIN_COLS);
    const dim3 block(FIN_COLS, FIN_SLICES);
    if (p->integral)
        finalize_kernel<true><<<grid, block, 0, s>>>(B, ld, partial, n_part, obj_now, best_obj, improved, st, p->ws.block_min,
                                                     trace_best, trace_ns, trace_cap, advance_t);
    else
        finalize_kernel<false><<<grid, block, 0, s>>>(B, ld, partial, n_part, obj_now, best_obj, improved, st, p->ws.block_min,
                                                      trace_best, trace_ns, trace_cap, advance_t);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status score_reduce(gda_problem* p, int32_t B, int32_t ld, const void* partial, int32_t n_part, double* obj,
                        cudaStream_t s) {
    return eval_finalize(p, B, ld, partial, n_part, obj, nullptr, nullptr, nullptr, nullptr, nullptr, 0, 0, s, nullptr);
}

// every row of the (padded) state, every column of the (padded) stride: improved[] is 0 for padding restarts
gda_status eval_commit(gda_problem* p, int32_t ld, const float* x, const int32_t* improved, uint8_t* x_bin,
                       cudaStream_t s, int64_t* launches) {
    const size_t n_vec = (size_t)p->n_pad * ld / 4;
    const unsigned grid = (unsigned)std::min<size_t>((n_vec + 255) / 256, (size_t)p->num_sms * 8);
    commit_kernel<<<grid, 256, 0, s>>>(n_vec, ld / 4, x, improved, p->ws.state, x_bin);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status eval_yg_partials(gda_problem* p, int32_t n_rows, int32_t B, const float* x, const float* y, float y_scalar, int32_t gfun,
                            float log_eps, double* partial, int32_t* n_part, cudaStream_t s) {
    (void)p;
    UpdParams up{};
    up.log_eps = log_eps; up.gfun = gfun;
    const dim3 grid((unsigned)((n_rows + 63) / 64), (unsigned)((B / 4 + 31) / 32));
    if (gfun == GDA_G_QUADRATIC) yg_partials_kernel<GDA_G_QUADRATIC><<<grid, 256, 0, s>>>(n_rows, B, x, y, y_scalar, up, partial);
    else yg_partials_kernel<GDA_G_ENTROPY><<<grid, 256, 0, s>>>(n_rows, B, x, y, y_scalar, up, partial);
    *n_part = (int32_t)grid.x;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status eval_xg_partials(gda_problem* p, int32_t ld, const float* x, const float* G, double* partial, int32_t* n_part, cudaStream_t s) {
    const dim3 grid((unsigned)((p->n + 63) / 64), (unsigned)((ld / 4 + 31) / 32));
    xg_partials_kernel<<<grid, 256, 0, s>>>(p->n, ld, x, G, p->d_cprime, partial);
    *n_part = (int32_t)grid.x;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status eval_sum_partials(int32_t B, int32_t ld, const double* partial, int32_t n_part, double* out, cudaStream_t s) {
    finalize_kernel<false><<<(unsigned)((B + FIN_COLS - 1) / FIN_COLS), dim3(FIN_COLS, FIN_SLICES), 0, s>>>(
        B, ld, partial, n_part, out, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0, 0);
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status eval_count_ones(gda_problem* p, int32_t B, const uint8_t* x_bin, int32_t* ones, cudaStream_t s, int64_t* launches) {
    count_ones_kernel<<<(unsigned)((B + 127) / 128), dim3(32, 32), 0, s>>>(p->n, B, p->ws.ld, x_bin, ones);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status eval_argbest(int32_t B, const double* obj, int32_t* best_restart, double* best_val,
                        cudaStream_t s, int64_t* launches) {
    argbest_kernel<<<1, 256, 0, s>>>(B, obj, best_restart, best_val);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}
