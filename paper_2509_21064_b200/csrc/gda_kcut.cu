// gda_kcut.cu -- PDBO on Max-k-Cut (Appendix B; readings K1-K5 of DESIGN.md).
//
//   min Tr(X W X^T) over one-hot columns X_{:,i};  X_{:,i} = SoftMax(Z_{:,i});  L = Tr(X W X^T) + sum_i y_i g(X_{:,i})
//   D_ji = dL/dX_ji = 2 (X W)_ji + y_i g'_j,   dL/dZ_ji = X_ji (D_ji - sum_l X_li D_li)        (softmax Jacobian)
//   Z+ = Z - alpha dL/dZ,   y+ = y + beta g(X_{:,i}),   X+ = SoftMax(Z+)
//
// Layout: Z and X are [k][n][B] fp32 planes (restart index contiguous), y and the labels [n][B].  One warp owns one
// (node, 128-restart chunk) item: the node's (col, 2 W) pairs are fetched once and broadcast by shuffle, and every
// neighbour is gathered from all k planes of X (k coalesced 512-byte requests), so the structure traffic and the
// address arithmetic are shared by the k SpMMs.  X is double-buffered (Jacobi), Z and y are updated in place; the
// update and the new softmax happen in registers.
#include "gda_internal.cuh"

#include <cstdlib>

namespace {

constexpr int WARPS = 8;
constexpr int THREADS = WARPS * 32;
constexpr int SW = 2;                // warps per block of the step kernel (Max-3-Cut n = 20000, B = 128: 29.4 us per step with 8, 28.25 with 4, 27.85 with 2)
constexpr int SCORE_ROWS = 64;

__device__ __forceinline__ float4 ld4c(const char* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

// SPLIT: one block of SPLIT_WARPS warps per (node, chunk); the warps take interleaved slices of 8 neighbours and warp 0 adds
// their sums in warp order and finishes the node.  Used when the launch would otherwise be a few warps per SM that each walk
// a long row (Max-3-Cut on the 800-node, degree-48 graph at the paper's B = 100: 800 warps, 12.95 -> see kcut_step).
constexpr int SPLIT_WARPS = 8, SPLIT_SLICE = 8;
template <int GFUN, int K, bool SPLIT = false>
__global__ void __launch_bounds__(32 * (SPLIT ? SPLIT_WARPS : SW))
kcut_step_kernel(int n, int B, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                 const float* __restrict__ val2, const float* __restrict__ x, float* __restrict__ z,
                 float* __restrict__ y, float* __restrict__ xn, UpdParams up) {
    __shared__ float4 red[SPLIT ? SPLIT_WARPS : 1][SPLIT ? K : 1][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int row = SPLIT ? blockIdx.x : blockIdx.x * SW + warp;
    if (row >= n) return;                                    // warp-uniform (SPLIT: block-uniform)
    const bool active = 4 * (blockIdx.y * 32 + lane) < B;
    const int c4 = active ? blockIdx.y * 32 + lane : B / 4 - 1;
    const uint32_t stride = 4u * (uint32_t)B;                // bytes per node row
    const uint64_t plane = (uint64_t)n * stride;             // bytes per part
    const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
    const int start = __ldg(rowptr + row), end = __ldg(rowptr + row + 1);

    float4 S[K];                                             // S_j = sum_l 2 W_il X_jl = dTr/dX_ji
#pragma unroll
    for (int j = 0; j < K; ++j) S[j] = make_float4(0.f, 0.f, 0.f, 0.f);
    constexpr int SLICE = SPLIT ? SPLIT_SLICE : 32, STEP = SPLIT ? SPLIT_SLICE * SPLIT_WARPS : 32;
    for (int base = start + (SPLIT ? SLICE * warp : 0); base < end; base += STEP) {
        const int cnt = min(SLICE, end - base);
        const int e = base + lane;
        const int my_c = lane < cnt ? __ldg(col + e) : 0;
        const float my_v = lane < cnt ? __ldg(val2 + e) : 0.0f;
        for (int u = 0; u < cnt; u += 2) {                   // two neighbours x K planes in flight; past the end: value 0
            const int c0 = __shfl_sync(0xffffffffu, my_c, u), c1 = __shfl_sync(0xffffffffu, my_c, min(u + 1, 31));
            const float v0 = __shfl_sync(0xffffffffu, my_v, u);
            const float v1 = u + 1 < cnt ? __shfl_sync(0xffffffffu, my_v, min(u + 1, 31)) : 0.0f;
            float4 g0[K], g1[K];
#pragma unroll
            for (int j = 0; j < K; ++j) {
                g0[j] = ld4c(xb + j * plane + (uint64_t)(uint32_t)c0 * stride);
                g1[j] = ld4c(xb + j * plane + (uint64_t)(uint32_t)c1 * stride);
            }
#pragma unroll
            for (int j = 0; j < K; ++j) {
                S[j].x = fmaf(v0, g0[j].x, S[j].x); S[j].y = fmaf(v0, g0[j].y, S[j].y);
                S[j].z = fmaf(v0, g0[j].z, S[j].z); S[j].w = fmaf(v0, g0[j].w, S[j].w);
                S[j].x = fmaf(v1, g1[j].x, S[j].x); S[j].y = fmaf(v1, g1[j].y, S[j].y);
                S[j].z = fmaf(v1, g1[j].z, S[j].z); S[j].w = fmaf(v1, g1[j].w, S[j].w);
            }
        }
    }

    // the node's own X, Z, y (SPLIT: warp 0 has them in flight while it waits for the other warps' sums)
    const size_t off = (size_t)row * B + 4 * c4;
    const size_t pl = (size_t)n * B;
    float4 X[K], Z[K];
    float4 yv = make_float4(0.f, 0.f, 0.f, 0.f);
    if (!SPLIT || warp == 0) {
#pragma unroll
        for (int j = 0; j < K; ++j) { X[j] = ldg4(x + j * pl + off); Z[j] = *reinterpret_cast<const float4*>(z + j * pl + off); }
        yv = *reinterpret_cast<const float4*>(y + off);
    }
    if (SPLIT) {
#pragma unroll
        for (int j = 0; j < K; ++j) red[warp][j][lane] = S[j];
        __syncthreads();
        if (warp != 0) return;
#pragma unroll
        for (int j = 0; j < K; ++j) {
            float4 t = red[0][j][lane];
            for (int w = 1; w < SPLIT_WARPS; ++w) { const float4 r = red[w][j][lane]; t.x += r.x; t.y += r.y; t.z += r.z; t.w += r.w; }
            S[j] = t;
        }
    }

    // per component (restart): g, D, the softmax chain rule, the step, the new softmax
    float4 yo;
#define KCUT_COMPONENT(F)                                                                              \
    {                                                                                                  \
        float gv = 0.0f, mean = 0.0f, D[K];                                                            \
        _Pragma("unroll") for (int j = 0; j < K; ++j) {                                                \
            const float v = X[j].F;                                                                    \
            float gp;                                                                                  \
            if (GFUN == GDA_G_QUADRATIC) { gv = fmaf(v, v, gv); gp = 2.0f * v; }                       \
            else { const float lg = fast_ln(fmaxf(v, up.log_eps)); gv = fmaf(v, v > 0.0f ? lg : 0.0f, gv); gp = lg + 1.0f; } \
            D[j] = fmaf(yv.F, gp, S[j].F);                                                             \
            mean = fmaf(v, D[j], mean);                                                                \
        }                                                                                              \
        if (GFUN == GDA_G_QUADRATIC) gv -= 1.0f;                                                       \
        yo.F = fmaf(up.beta, gv, yv.F);                                                                \
        float zmax = -3.0e38f;                                                                         \
        _Pragma("unroll") for (int j = 0; j < K; ++j) {                                                \
            Z[j].F = Z[j].F - up.alpha * (X[j].F * (D[j] - mean));                                     \
            zmax = fmaxf(zmax, Z[j].F);                                                                \
        }                                                                                              \
        float sum = 0.0f;                                                                              \
        _Pragma("unroll") for (int j = 0; j < K; ++j) { X[j].F = __expf(Z[j].F - zmax); sum += X[j].F; } \
        const float inv = 1.0f / sum;                                                                  \
        _Pragma("unroll") for (int j = 0; j < K; ++j) X[j].F *= inv;                                   \
    }
    KCUT_COMPONENT(x) KCUT_COMPONENT(y) KCUT_COMPONENT(z) KCUT_COMPONENT(w)
#undef KCUT_COMPONENT
    if (!active) return;
#pragma unroll
    for (int j = 0; j < K; ++j) {
        *reinterpret_cast<float4*>(z + j * pl + off) = Z[j];
        *reinterpret_cast<float4*>(xn + j * pl + off) = X[j];
    }
    *reinterpret_cast<float4*>(y + off) = yo;
}

// X = SoftMax(Z) column by column (start of a run)
__global__ void __launch_bounds__(256)
kcut_softmax_kernel(size_t n_vec, size_t pl, int k, const float* __restrict__ z, float* __restrict__ x) {
    const size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n_vec) return;
    float4 m = *reinterpret_cast<const float4*>(z + 4 * v);
    for (int j = 1; j < k; ++j) {
        const float4 t = *reinterpret_cast<const float4*>(z + j * pl + 4 * v);
        m.x = fmaxf(m.x, t.x); m.y = fmaxf(m.y, t.y); m.z = fmaxf(m.z, t.z); m.w = fmaxf(m.w, t.w);
    }
    float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int j = 0; j < k; ++j) {
        const float4 t = *reinterpret_cast<const float4*>(z + j * pl + 4 * v);
        const float4 e = make_float4(__expf(t.x - m.x), __expf(t.y - m.y), __expf(t.z - m.z), __expf(t.w - m.w));
        s.x += e.x; s.y += e.y; s.z += e.z; s.w += e.w;
        *reinterpret_cast<float4*>(x + j * pl + 4 * v) = e;
    }
    for (int j = 0; j < k; ++j) {
        float4 e = *reinterpret_cast<float4*>(x + j * pl + 4 * v);
        e.x /= s.x; e.y /= s.y; e.z /= s.z; e.w /= s.w;
        *reinterpret_cast<float4*>(x + j * pl + 4 * v) = e;
    }
}

// labels[i][b] = argmax_j Z[j][i][b], lowest j on ties (reading K4)
__global__ void __launch_bounds__(256)
kcut_label_kernel(size_t n_vec, size_t pl, int k, const float* __restrict__ z, uint8_t* __restrict__ lab) {
    const size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n_vec) return;
    float4 m = *reinterpret_cast<const float4*>(z + 4 * v);
    uchar4 a = make_uchar4(0, 0, 0, 0);
    for (int j = 1; j < k; ++j) {
        const float4 t = *reinterpret_cast<const float4*>(z + j * pl + 4 * v);
        if (t.x > m.x) { m.x = t.x; a.x = (uint8_t)j; }
        if (t.y > m.y) { m.y = t.y; a.y = (uint8_t)j; }
        if (t.z > m.z) { m.z = t.z; a.z = (uint8_t)j; }
        if (t.w > m.w) { m.w = t.w; a.w = (uint8_t)j; }
    }
    *reinterpret_cast<uchar4*>(lab + 4 * v) = a;
}

// S5: partial[rb][b] = sum over the rows i of block rb and their entries l of W_il [label_i == label_l] = Tr(Xh W Xh^T)
template <bool INTEGRAL>
__global__ void __launch_bounds__(THREADS)
kcut_score_kernel(int n, int B, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                  const float* __restrict__ val2, const uint8_t* __restrict__ lab, void* __restrict__ partial) {
    using acc_t = typename std::conditional<INTEGRAL, long long, double>::type;
    __shared__ acc_t red[WARPS][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c4 = blockIdx.y * 32 + lane;
    const bool active = 4 * c4 < B;
    acc_t acc[4] = {0, 0, 0, 0};
    for (int r = warp; r < SCORE_ROWS; r += WARPS) {
        const int row = blockIdx.x * SCORE_ROWS + r;
        if (row >= n) break;
        const int start = __ldg(rowptr + row), end = __ldg(rowptr + row + 1);
        const uchar4 mine = active ? *reinterpret_cast<const uchar4*>(lab + (size_t)row * B + 4 * c4) : make_uchar4(0, 0, 0, 0);
        float s[4] = {0.f, 0.f, 0.f, 0.f};
        int si[4] = {0, 0, 0, 0};
        for (int base = start; base < end; base += 32) {
            const int e = base + lane;
            const int my_c = e < end ? __ldg(col + e) : 0;
            const float my_v = e < end ? __ldg(val2 + e) : 0.0f;
            const int cnt = min(32, end - base);
            for (int u = 0; u < cnt; ++u) {
                const int c = __shfl_sync(0xffffffffu, my_c, u);
                const float v = __shfl_sync(0xffffffffu, my_v, u);
                if (!active) continue;
                const uchar4 o = *reinterpret_cast<const uchar4*>(lab + (size_t)c * B + 4 * c4);
                if (INTEGRAL) {
                    const int vi = __float2int_rn(v);
                    si[0] += o.x == mine.x ? vi : 0; si[1] += o.y == mine.y ? vi : 0;
                    si[2] += o.z == mine.z ? vi : 0; si[3] += o.w == mine.w ? vi : 0;
                } else {
                    s[0] += o.x == mine.x ? v : 0.f; s[1] += o.y == mine.y ? v : 0.f;
                    s[2] += o.z == mine.z ? v : 0.f; s[3] += o.w == mine.w ? v : 0.f;
                }
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (INTEGRAL) acc[q] += (long long)(si[q] / 2);   // val2 = 2 W_il: even
            else acc[q] += 0.5 * (double)s[q];
        }
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) red[warp][lane][q] = acc[q];
    __syncthreads();
    if (warp == 0 && active) {
        acc_t* out = reinterpret_cast<acc_t*>(partial) + (size_t)blockIdx.x * B + 4 * c4;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            acc_t t = red[0][lane][q];
            for (int w = 1; w < WARPS; ++w) t += red[w][lane][q];
            out[q] = t;
        }
    }
}

// best-so-far labels: x_bin[:, b] = lab[:, b] for every restart whose objective improved at this evaluation
__global__ void __launch_bounds__(256)
kcut_commit_kernel(size_t n_vec, int B4, const uint8_t* __restrict__ lab, const int32_t* __restrict__ improved,
                   const RunState* __restrict__ st, uint8_t* __restrict__ x_bin) {
    if (st->any_improved == 0u) return;                      // no restart improved at this evaluation (finalize_kernel)
    const size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n_vec) return;
    const int b0 = 4 * (int)(v % (size_t)B4);
    const uchar4 nw = *reinterpret_cast<const uchar4*>(lab + 4 * v);
    uchar4 cur = *reinterpret_cast<uchar4*>(x_bin + 4 * v);
    if (improved[b0 + 0]) cur.x = nw.x;
    if (improved[b0 + 1]) cur.y = nw.y;
    if (improved[b0 + 2]) cur.z = nw.z;
    if (improved[b0 + 3]) cur.w = nw.w;
    *reinterpret_cast<uchar4*>(x_bin + 4 * v) = cur;
}

template <int GFUN>
void launch_k(gda_problem* p, int32_t B, dim3 grid, const float* x, float* z, float* y, float* xn, const UpdParams& up,
              cudaStream_t s) {
    // few warps that each walk a long row: split the rows (the rule of the sparse QUBO path, gda_sparse.cu)
    const bool split = p->opt_split_all >= 0 ? p->opt_split_all == 1      // GDA_OPT_SPLIT_ALL_ROWS
                                 : (int64_t)p->n * grid.y < (int64_t)p->num_sms * 12 && p->nnz >= 16 * (int64_t)p->n;
#define KCUT_CASE(K) case K: if (split) kcut_step_kernel<GFUN, K, true><<<dim3((unsigned)p->n, grid.y), 32 * SPLIT_WARPS, 0, s>>>(p->n, B, p->d_rowptr, p->d_col, p->d_val2, x, z, y, xn, up); \
                             else kcut_step_kernel<GFUN, K><<<grid, 32 * SW, 0, s>>>(p->n, B, p->d_rowptr, p->d_col, p->d_val2, x, z, y, xn, up); break;
    switch (p->kparts) { KCUT_CASE(2) KCUT_CASE(3) KCUT_CASE(4) KCUT_CASE(5) KCUT_CASE(6) KCUT_CASE(7) KCUT_CASE(8) default: break; }
#undef KCUT_CASE
}

}  // namespace

gda_status kcut_step(gda_problem* p, int32_t B, const float* x, float* z, float* y, float* xn, const UpdParams& up,
                     cudaStream_t s, int64_t* launches) {
    const dim3 grid((unsigned)((p->n + SW - 1) / SW), (unsigned)((B / 4 + 31) / 32));
    if (up.gfun == GDA_G_QUADRATIC) launch_k<GDA_G_QUADRATIC>(p, B, grid, x, z, y, xn, up, s);
    else launch_k<GDA_G_ENTROPY>(p, B, grid, x, z, y, xn, up, s);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status kcut_softmax(gda_problem* p, int32_t B, const float* z, float* x, cudaStream_t s, int64_t* launches) {
    const size_t pl = (size_t)p->n * B, n_vec = pl / 4;
    kcut_softmax_kernel<<<(unsigned)((n_vec + 255) / 256), 256, 0, s>>>(n_vec, pl, p->kparts, z, x);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

int32_t kcut_num_partials(const gda_problem* p, int32_t) { return (p->n + SCORE_ROWS - 1) / SCORE_ROWS; }

gda_status kcut_score_partials(gda_problem* p, int32_t B, const float* z, uint8_t* lab, void* partial, int32_t* n_part,
                               cudaStream_t s, int64_t* launches) {
    const size_t pl = (size_t)p->n * B, n_vec = pl / 4;
    kcut_label_kernel<<<(unsigned)((n_vec + 255) / 256), 256, 0, s>>>(n_vec, pl, p->kparts, z, lab);
    const dim3 grid((unsigned)kcut_num_partials(p, B), (unsigned)((B / 4 + 31) / 32));
    if (p->integral) kcut_score_kernel<true><<<grid, THREADS, 0, s>>>(p->n, B, p->d_rowptr, p->d_col, p->d_val2, lab, partial);
    else kcut_score_kernel<false><<<grid, THREADS, 0, s>>>(p->n, B, p->d_rowptr, p->d_col, p->d_val2, lab, partial);
    if (launches) *launches += 2;
    *n_part = (int32_t)grid.x;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

// gda_grad / gda_lagrangian for Max-k-Cut (not on the hot path: plain warp-per-node loops, k at run time).
//   MODE 0: G[j][i][b] = X_ji (D_ji - sum_l X_li D_li), D = 2 X W: grad_Z of Tr(X W X^T) at X = SoftMax(Z)
//   MODE 1: partial[rb][b] = sum over the nodes i of block rb of  sum_j X_ji (X W)_ji + y_i g(X_:,i)
static __device__ __forceinline__ void fma4(float4& a, float v, const float4& g) {
    a.x = fmaf(v, g.x, a.x); a.y = fmaf(v, g.y, a.y); a.z = fmaf(v, g.z, a.z); a.w = fmaf(v, g.w, a.w);
}
template <int MODE>
__global__ void __launch_bounds__(THREADS)
kcut_aux_kernel(int n, int B, int k, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                const float* __restrict__ val2, const float* __restrict__ x, const float* __restrict__ y, float y_scalar,
                int gfun, float* __restrict__ G, double* __restrict__ partial) {
    __shared__ double red[MODE == 1 ? WARPS : 1][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c4 = blockIdx.y * 32 + lane;
    const bool active = 4 * c4 < B;
    const size_t pl = (size_t)n * B;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int r = warp; r < SCORE_ROWS && active; r += WARPS) {
        const int row = blockIdx.x * SCORE_ROWS + r;
        if (row >= n) break;
        const size_t off = (size_t)row * B + 4 * c4;
        float4 S[8], X[8];
        for (int j = 0; j < k; ++j) { S[j] = make_float4(0.f, 0.f, 0.f, 0.f); X[j] = ldg4(x + j * pl + off); }
        for (int a = __ldg(rowptr + row); a < __ldg(rowptr + row + 1); ++a) {
            const int c = __ldg(col + a);
            const float v = __ldg(val2 + a);
            for (int j = 0; j < k; ++j) fma4(S[j], v, ldg4(x + j * pl + (size_t)c * B + 4 * c4));
        }
        if (MODE == 0) {
            float4 mean = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int j = 0; j < k; ++j) { mean.x = fmaf(X[j].x, S[j].x, mean.x); mean.y = fmaf(X[j].y, S[j].y, mean.y); mean.z = fmaf(X[j].z, S[j].z, mean.z); mean.w = fmaf(X[j].w, S[j].w, mean.w); }
            for (int j = 0; j < k; ++j)
                *reinterpret_cast<float4*>(G + j * pl + off) = make_float4(X[j].x * (S[j].x - mean.x), X[j].y * (S[j].y - mean.y),
                                                                          X[j].z * (S[j].z - mean.z), X[j].w * (S[j].w - mean.w));
        } else {
            const float4 yv = y ? *reinterpret_cast<const float4*>(y + off) : make_float4(y_scalar, y_scalar, y_scalar, y_scalar);
            const float yq[4] = {yv.x, yv.y, yv.z, yv.w};
            for (int q = 0; q < 4; ++q) {
                double tr = 0.0, g = 0.0;
                for (int j = 0; j < k; ++j) {
                    const float v = q == 0 ? X[j].x : q == 1 ? X[j].y : q == 2 ? X[j].z : X[j].w;
                    const float sv = q == 0 ? S[j].x : q == 1 ? S[j].y : q == 2 ? S[j].z : S[j].w;
                    tr += 0.5 * (double)v * (double)sv;                      // val2 = 2 W_il
                    if (gfun == GDA_G_QUADRATIC) g += (double)v * (double)v;
                    else if (v > 0.0f) g += (double)v * (double)logf(v);
                }
                if (gfun == GDA_G_QUADRATIC) g -= 1.0;
                acc[q] += tr + (double)yq[q] * g;
            }
        }
    }
    if (MODE == 1) {
#pragma unroll
        for (int q = 0; q < 4; ++q) red[warp][lane][q] = acc[q];
        __syncthreads();
        if (warp == 0 && active) {
            double* out = partial + (size_t)blockIdx.x * B + 4 * c4;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                double t = red[0][lane][q];
                for (int w = 1; w < WARPS; ++w) t += red[w][lane][q];
                out[q] = t;
            }
        }
    }
}

gda_status kcut_grad(gda_problem* p, int32_t B, const float* x, float* G, cudaStream_t s) {
    const dim3 grid((unsigned)kcut_num_partials(p, B), (unsigned)((B / 4 + 31) / 32));
    kcut_aux_kernel<0><<<grid, THREADS, 0, s>>>(p->n, B, p->kparts, p->d_rowptr, p->d_col, p->d_val2, x, nullptr, 0.0f, 0, G, nullptr);
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status kcut_value_partials(gda_problem* p, int32_t B, const float* x, const float* y, float y_scalar, int32_t gfun,
                               double* partial, int32_t* n_part, cudaStream_t s) {
    const dim3 grid((unsigned)kcut_num_partials(p, B), (unsigned)((B / 4 + 31) / 32));
    kcut_aux_kernel<1><<<grid, THREADS, 0, s>>>(p->n, B, p->kparts, p->d_rowptr, p->d_col, p->d_val2, x, y, y_scalar, gfun, nullptr, partial);
    *n_part = (int32_t)grid.x;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status kcut_commit(gda_problem* p, int32_t B, const uint8_t* lab, const int32_t* improved, uint8_t* x_bin,
                       cudaStream_t s, int64_t* launches) {
    const size_t n_vec = (size_t)p->n * B / 4;
    kcut_commit_kernel<<<(unsigned)((n_vec + 255) / 256), 256, 0, s>>>(n_vec, B / 4, lab, improved, p->ws.state, x_bin);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}
