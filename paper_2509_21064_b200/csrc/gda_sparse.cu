// gda_sparse.cu -- S1 + S4 for sparse QUBO / Max-Cut: batched CSR SpMM gradient fused with the GDA update.
//
//   G = 2 Q_off X + c' 1^T            (multilinear extension of x^T Q x + c^T x)
//   x+ = clip(x - alpha (G + y g'(x))),  y+ = y + beta g(x),  perturbation near 1/2
//
// Layout: X, Y are [n][B] fp32 with the restart index contiguous, so the gather of row j for 128
// consecutive restarts is one coalesced 512-byte request (a float4 per lane).  One warp owns one
// (row, 128-restart chunk) item: it loads the row's (col, val) pairs with one coalesced load and
// broadcasts them by shuffle, gathers, and applies the fused update in registers -- G never goes to memory.
// Rows with more than HEAVY_DEG non-zeros are split across the 8 warps of a block (row-split variant).
#include "gda_internal.cuh"

namespace {

constexpr int WARPS = 8;
constexpr int THREADS = WARPS * 32;
constexpr int HEAVY_DEG = 256;     // rows above this use the row-split kernel
constexpr int SCORE_ROWS = 64;     // most rows per block in the scoring kernels (fewer when that leaves SMs idle)

__device__ __forceinline__ void fma4(float4& a, float v, const float4& g) {
    a.x = fmaf(v, g.x, a.x); a.y = fmaf(v, g.y, a.y); a.z = fmaf(v, g.z, a.z); a.w = fmaf(v, g.w, a.w);
}

// One 512-byte gather: row c of X for this lane's four restarts.  xb = X + this lane's column offset (bytes),
// stride = 4 B bytes per row; c * stride is one IMAD.WIDE.U32 (no 64-bit shifts and carries per gather).
__device__ __forceinline__ float4 gather4(const char* __restrict__ xb, uint32_t stride, int c) {
    return __ldg(reinterpret_cast<const float4*>(xb + (uint64_t)(uint32_t)c * (uint64_t)stride));
}

// acc += sum_{u < cnt} v_u * X[c_u][this lane's columns], where entry u's column is held by lane c_lane0 + u (in
// word_c) and its value by lane v_lane0 + u (in word_v): broadcast by shuffle, 4 independent 512 B gathers in flight.
// Every lane takes part with a VALID column offset (lanes past a ragged B are clamped by the caller and only their
// stores are suppressed), so nothing here is predicated on "active".
__device__ __forceinline__ void accumulate_lanes(float4& acc, int word_c, int c_lane0, int word_v, int v_lane0, int cnt,
                                                 const char* __restrict__ xb, uint32_t stride) {
    for (int u = 0; u < cnt; u += 4) {
        int c[4]; float v[4]; float4 g[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {                        // past the end: the last entry again (same line) with value 0
            const int e = min(u + q, cnt - 1);
            c[q] = __shfl_sync(0xffffffffu, word_c, c_lane0 + e);
            v[q] = __int_as_float(__shfl_sync(0xffffffffu, word_v, v_lane0 + e));
            if (u + q >= cnt) v[q] = 0.0f;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) g[q] = gather4(xb, stride, c[q]);
#pragma unroll
        for (int q = 0; q < 4; ++q) fma4(acc, v[q], g[q]);
    }
}

// sum_k val2[k] * X[col[k]][this lane's columns]  for k in [start, end): (col,val) fetched 32 at a time, one per lane
__device__ __forceinline__ float4 gather_row(const int32_t* __restrict__ col, const float* __restrict__ val2,
                                             int start, int end, const char* __restrict__ xb, uint32_t stride, int lane) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int base = start; base < end; base += 32) {
        const int k = base + lane;
        const int my_c = (k < end) ? __ldg(col + k) : 0;
        const int my_v = (k < end) ? __ldg(reinterpret_cast<const int*>(val2) + k) : 0;
        accumulate_lanes(acc, my_c, 0, my_v, 0, min(32, end - base), xb, stride);
    }
    return acc;
}

// S4 for one (row, float4 of restarts).  DUAL (PDBO-s): `mu` is this step's multiplier for the four restarts, y is
// not touched, and the values of g(x^t) are returned in gs (0 for lanes past a ragged B).
template <int GFUN, bool DUAL>
__device__ __forceinline__ void update_store(int row, int c4, int B, bool active, float4 G, const float* __restrict__ x,
                                             float* __restrict__ y, float* __restrict__ xn,
                                             const UpdParams& up, uint32_t t, float4 mu, float4& gs) {
    const size_t off = (size_t)row * B + 4 * c4;
    const float4 xv = ldg4(x + off);
    const float4 yv = DUAL ? mu : *reinterpret_cast<const float4*>(y + off);
    float4 xo, yo;
    gda_update4<GFUN>(xv, yv, G, up, t, (uint32_t)row, 4u * (uint32_t)c4, xo, yo);
    if (!active) return;
    *reinterpret_cast<float4*>(xn + off) = xo;
    if (DUAL) gs = make_float4(gda_g<GFUN>(xv.x, up), gda_g<GFUN>(xv.y, up), gda_g<GFUN>(xv.z, up), gda_g<GFUN>(xv.w, up));
    else *reinterpret_cast<float4*>(y + off) = yo;
}

// warp-per-(row, 128-restart chunk): blockIdx.y = chunk, the block's 8 warps take 8 consecutive rows.
// MODE 0: fused step, MODE 1: write G only (gda_grad).
// ELL: rows of degree <= 8 come as one packed 64-byte record (8 columns, 8 values; gda_api.cu) fetched with a single
// coalesced load, which removes the rowptr -> (col, val) hop from the dependent chain of a row; a record whose word 0
// is -1 sends the row through its CSR entries.  40 registers (6 blocks per SM).  Measured on config 3 (profiles/):
// 17.3 us per step before, 16.3 us with the lean gather loop, 14.8 us with the records and 6 blocks per SM;
// prefetching the row's own x, y lines into L1 up front was slower (15.1 us) and is not done.
// DUAL (PDBO-s, MODE 0 only): the multiplier is one number per restart (sd.mu), y is not read or written, and the
// block leaves the sum of g(x_i^t) over its rows in sd.gpart[blockIdx.x].
template <int GFUN, int MODE, bool ELL, bool DUAL>
__global__ void __launch_bounds__(THREADS, 6)
spmm_step_warp(int n_rows, const int32_t* __restrict__ row_list, int B,
               const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
               const float* __restrict__ val2, const int32_t* __restrict__ ell, const float* __restrict__ cprime,
               const float* __restrict__ x, float* __restrict__ y, float* __restrict__ xn,
               UpdParams up, ScalarDual sd, const RunState* __restrict__ st, uint32_t t_off) {
    __shared__ float4 gred[DUAL ? WARPS : 1][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ridx = blockIdx.x * WARPS + warp;
    const bool active = 4 * (blockIdx.y * 32 + lane) < B;
    const int c4 = active ? blockIdx.y * 32 + lane : B / 4 - 1;      // ragged B: idle lanes recompute the last float4
    if (DUAL) {
        float4 gs = make_float4(0.f, 0.f, 0.f, 0.f), mu = ldg4(sd.mu + 4 * c4);
        if (ridx < n_rows) {                                 // warp-uniform
            const int row = row_list ? __ldg(row_list + ridx) : ridx;
            const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
            const uint32_t stride = 4u * (uint32_t)B;
            float4 G = make_float4(0.f, 0.f, 0.f, 0.f);
            bool csr = true;
            if (ELL) {
                const int w = __ldg(ell + (size_t)row * 16 + (lane & 15));
                csr = __shfl_sync(0xffffffffu, w, 0) < 0;
                if (!csr) accumulate_lanes(G, w, 0, w, 8, __popc(__ballot_sync(0xffffffffu, w != 0 && (lane & 24) == 8)), xb, stride);
            }
            if (csr) G = gather_row(col, val2, __ldg(rowptr + row), __ldg(rowptr + row + 1), xb, stride, lane);
            const float cp = __ldg(cprime + row);
            G.x += cp; G.y += cp; G.z += cp; G.w += cp;
            update_store<GFUN, true>(row, c4, B, active, G, x, y, xn, up, (st ? st->t : 0u) + t_off, mu, gs);
        }
        scalar_dual_block_sum<WARPS>(gs, gred, warp, lane, active, sd.gpart + (size_t)blockIdx.x * B + 4 * c4);
        return;
    }
    if (ridx >= n_rows) return;                              // warp-uniform
    const int row = row_list ? __ldg(row_list + ridx) : ridx;
    const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
    const uint32_t stride = 4u * (uint32_t)B;
    float4 G = make_float4(0.f, 0.f, 0.f, 0.f);
    bool csr = true;
    if (ELL) {
        const int w = __ldg(ell + (size_t)row * 16 + (lane & 15));
        csr = __shfl_sync(0xffffffffu, w, 0) < 0;
        if (!csr) {
            const int cnt = __popc(__ballot_sync(0xffffffffu, w != 0 && (lane & 24) == 8));   // values sit in lanes 8..15
            accumulate_lanes(G, w, 0, w, 8, cnt, xb, stride);
        }
    }
    if (csr) G = gather_row(col, val2, __ldg(rowptr + row), __ldg(rowptr + row + 1), xb, stride, lane);
    const float cp = __ldg(cprime + row);
    G.x += cp; G.y += cp; G.z += cp; G.w += cp;
    if (MODE == 1) { if (active) *reinterpret_cast<float4*>(xn + (size_t)row * B + 4 * c4) = G; return; }
    const uint32_t t = (st ? st->t : 0u) + t_off;
    float4 unused;
    update_store<GFUN, false>(row, c4, B, active, G, x, y, xn, up, t, make_float4(0.f, 0.f, 0.f, 0.f), unused);
}

// ---- narrow variant for few restarts (B <= 64; the paper's own runs use B = 10, Table 6) ---------------------------
// With one warp per (row, 128-restart chunk) only B / 4 of the 32 lanes have work when B is small (3 lanes at B = 12).
// Here G = the smallest power of two >= B / 4 lanes serve one row and a warp takes 32 / G rows at once: lane = (row in
// the warp, float4 of restarts).  Every lane walks its OWN row's entries (the loads of (col, val) are broadcasts inside
// its lane group), four gathers in flight, up to the longest row of the warp with the shorter rows predicated off.
template <int GFUN, int G>
__global__ void __launch_bounds__(THREADS)
spmm_step_narrow(int n, int B, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                 const float* __restrict__ val2, const float* __restrict__ cprime, const float* __restrict__ x,
                 float* __restrict__ y, float* __restrict__ xn, UpdParams up, const RunState* __restrict__ st, uint32_t t_off) {
    constexpr int R = 32 / G;                                // rows per warp
    const int lane = threadIdx.x & 31;
    const int row_raw = (blockIdx.x * WARPS + (threadIdx.x >> 5)) * R + lane / G;
    const int cl = lane % G;
    const bool active = row_raw < n && 4 * cl < B;
    const int row = min(row_raw, n - 1);                     // idle lanes recompute a valid element, only stores are suppressed
    const int c4 = 4 * cl < B ? cl : 0;
    const int start = __ldg(rowptr + row);
    const int deg = row_raw < n ? __ldg(rowptr + row + 1) - start : 0;
    int maxdeg = deg;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) maxdeg = max(maxdeg, __shfl_xor_sync(0xffffffffu, maxdeg, o));
    const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
    const uint32_t stride = 4u * (uint32_t)B;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int a = 0; a < maxdeg; a += 4) {
        int c[4]; float v[4]; float4 g[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {                        // past the row's end: (own row, 0)
            const bool ok = a + q < deg;
            c[q] = ok ? __ldg(col + start + a + q) : row;
            v[q] = ok ? __ldg(val2 + start + a + q) : 0.0f;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) g[q] = gather4(xb, stride, c[q]);
#pragma unroll
        for (int q = 0; q < 4; ++q) fma4(acc, v[q], g[q]);
    }
    const float cp = __ldg(cprime + row);
    acc.x += cp; acc.y += cp; acc.z += cp; acc.w += cp;
    float4 unused;
    update_store<GFUN, false>(row, c4, B, active, acc, x, y, xn, up, (st ? st->t : 0u) + t_off, make_float4(0.f, 0.f, 0.f, 0.f), unused);
}

// row-split: one block per (heavy row, chunk); the 8 warps take interleaved 32-entry slices of the row
// DUAL: as above; the row's g values go to sd.gpart[gpart_row0 + ridx].
template <int GFUN, int MODE, bool DUAL>
__global__ void __launch_bounds__(THREADS)
spmm_step_split(int n_rows, const int32_t* __restrict__ row_list, int B, int chunks,
                const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                const float* __restrict__ val2, const float* __restrict__ cprime,
                const float* __restrict__ x, float* __restrict__ y, float* __restrict__ xn,
                UpdParams up, ScalarDual sd, int gpart_row0, const RunState* __restrict__ st, uint32_t t_off) {
    __shared__ float4 red[WARPS][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ridx = blockIdx.x / chunks, chunk = blockIdx.x % chunks;
    const int row = __ldg(row_list + ridx);
    const bool active = 4 * (chunk * 32 + lane) < B;
    const int c4 = active ? chunk * 32 + lane : B / 4 - 1;
    const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
    const int start = __ldg(rowptr + row), end = __ldg(rowptr + row + 1);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int base = start + 32 * warp; base < end; base += 32 * WARPS) {
        const float4 part = gather_row(col, val2, base, min(base + 32, end), xb, 4u * (uint32_t)B, lane);
        acc.x += part.x; acc.y += part.y; acc.z += part.z; acc.w += part.w;
    }
    red[warp][lane] = acc;
    __syncthreads();
    if (warp != 0) return;
    float4 G = red[0][lane];
#pragma unroll
    for (int w = 1; w < WARPS; ++w) { const float4 r = red[w][lane]; G.x += r.x; G.y += r.y; G.z += r.z; G.w += r.w; }
    const float cp = __ldg(cprime + row);
    G.x += cp; G.y += cp; G.z += cp; G.w += cp;
    if (MODE == 1) { if (active) *reinterpret_cast<float4*>(xn + (size_t)row * B + 4 * c4) = G; return; }
    const uint32_t t = (st ? st->t : 0u) + t_off;
    float4 gs = make_float4(0.f, 0.f, 0.f, 0.f), mu = gs;
    if (DUAL) {
        mu = ldg4(sd.mu + 4 * c4);
    }
    update_store<GFUN, DUAL>(row, c4, B, active, G, x, y, xn, up, t, mu, gs);
    if (DUAL && active) *reinterpret_cast<float4*>(sd.gpart + (size_t)(gpart_row0 + ridx) * B + 4 * c4) = gs;
}

// ---- resident variant for tiny problems (config 1: n = 20, B = 64) -----------------------------------------------
// When the whole state and the CSR fit one block's shared memory (n B <= RESIDENT_MAX elements: x double-buffered and
// y, 12 bytes per element), a chunk of `len` GDA steps is ONE launch of one block: the iterates stay in shared memory, steps are
// separated by __syncthreads(), and only the last iterate goes back to global memory.  Config 1: 1.4 us per step
// (one SM's issue rate: about 3000 warp instructions per step) instead of 2.2 us per kernel launch.  The arithmetic per element is that of spmm_step_warp (same
// order of the row's entries, same fused update).
constexpr int RESIDENT_MAX = 12288;
constexpr int RESIDENT_THREADS = 1024;
constexpr int RESIDENT_SMEM = 200 * 1024;         // state + the whole CSR

template <int GFUN>
__global__ void __launch_bounds__(RESIDENT_THREADS)
spmm_steps_resident(int n, int B, int nnz, int len, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                    const float* __restrict__ val2, const float* __restrict__ cprime, const float* __restrict__ x_in,
                    float* __restrict__ y, float* __restrict__ x_out, UpdParams up, const RunState* __restrict__ st) {
    extern __shared__ float sm[];
    const int total = n * B;
    float* xa = sm;                                          // x^t and x^{t+1} alternate between xa and xb
    float* xb = sm + total;
    float* ys = sm + 2 * total;
    float* cps = ys + total;                                 // c'[n]
    float* vs = cps + n;                                     // val2[nnz]
    int* cs = reinterpret_cast<int*>(vs + nnz);              // col[nnz]
    int* rp = cs + nnz;                                      // rowptr[n + 1]
    for (int e = threadIdx.x; e < total; e += RESIDENT_THREADS) { xa[e] = x_in[e]; ys[e] = y[e]; }
    for (int e = threadIdx.x; e < nnz; e += RESIDENT_THREADS) { vs[e] = val2[e]; cs[e] = col[e] * B; }
    for (int e = threadIdx.x; e <= n; e += RESIDENT_THREADS) { rp[e] = rowptr[e]; if (e < n) cps[e] = cprime[e]; }
    __syncthreads();
    const uint32_t t0 = st ? st->t : 0u;
    for (int k = 0; k < len; ++k) {
        for (int e = threadIdx.x; e < total; e += RESIDENT_THREADS) {
            const int i = e / B, b = e - i * B;
            float acc = 0.0f;
            const int a1 = rp[i + 1];
#pragma unroll 4
            for (int a = rp[i]; a < a1; ++a) acc = fmaf(vs[a], xa[cs[a] + b], acc);     // loads of later entries issue early
            float xn, yn;
            gda_update<GFUN>(xa[e], ys[e], acc + cps[i], up, t0 + (uint32_t)k, (uint32_t)i, (uint32_t)b, xn, yn);
            xb[e] = xn;
            ys[e] = yn;
        }
        __syncthreads();
        float* tmp = xa; xa = xb; xb = tmp;
    }
    for (int e = threadIdx.x; e < total; e += RESIDENT_THREADS) { x_out[e] = xa[e]; y[e] = ys[e]; }
}

// S5 for sparse QUBO: partial[rb][b] = sum over the rows of block rb of x_hat_i ((Q_off x_hat)_i + c'_i)
template <bool INTEGRAL>
__global__ void __launch_bounds__(THREADS)
spmm_score(int n, int B, int rows_per_block, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
           const float* __restrict__ val2, const float* __restrict__ cprime, const float* __restrict__ x,
           void* __restrict__ partial) {
    using acc_t = typename std::conditional<INTEGRAL, long long, double>::type;
    __shared__ acc_t red[WARPS][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c4 = blockIdx.y * 32 + lane;
    const bool active = 4 * c4 < B;
    const int row0 = blockIdx.x * rows_per_block;
    acc_t acc[4] = {0, 0, 0, 0};
    for (int r = warp; r < rows_per_block; r += WARPS) {
        const int row = row0 + r;
        if (row >= n) break;
        const int start = __ldg(rowptr + row), end = __ldg(rowptr + row + 1);
        float s[4] = {0.f, 0.f, 0.f, 0.f};                   // fp32 row sums of val2 * x_hat_j
        int si[4] = {0, 0, 0, 0};
        for (int base = start; base < end; base += 32) {
            const int k = base + lane;
            const int my_c = (k < end) ? __ldg(col + k) : 0;
            const float my_v = (k < end) ? __ldg(val2 + k) : 0.0f;          // lanes past the end: (row 0, value 0)
            const int cnt = min(32, end - base);
            for (int u = 0; u < cnt; u += 4) {                               // 4 independent gathers in flight
                int c[4]; float v[4]; float4 g[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {                                // u + q <= 31
                    c[q] = __shfl_sync(0xffffffffu, my_c, u + q);
                    v[q] = __shfl_sync(0xffffffffu, my_v, u + q);
                }
                if (!active) continue;
#pragma unroll
                for (int q = 0; q < 4; ++q) g[q] = ldg4(x + (size_t)c[q] * B + 4 * c4);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    if (INTEGRAL) {
                        const int vi = __float2int_rn(v[q]);
                        si[0] += g[q].x > 0.5f ? vi : 0; si[1] += g[q].y > 0.5f ? vi : 0;
                        si[2] += g[q].z > 0.5f ? vi : 0; si[3] += g[q].w > 0.5f ? vi : 0;
                    } else {
                        s[0] += g[q].x > 0.5f ? v[q] : 0.f; s[1] += g[q].y > 0.5f ? v[q] : 0.f;
                        s[2] += g[q].z > 0.5f ? v[q] : 0.f; s[3] += g[q].w > 0.5f ? v[q] : 0.f;
                    }
                }
            }
        }
        if (!active) continue;
        const float4 xi = ldg4(x + (size_t)row * B + 4 * c4);
        const float cp = __ldg(cprime + row);
        const bool on[4] = {xi.x > 0.5f, xi.y > 0.5f, xi.z > 0.5f, xi.w > 0.5f};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (!on[q]) continue;
            if (INTEGRAL) acc[q] += (long long)(si[q] / 2) + (long long)__float2int_rn(cp);  // val2 = 2 Q_ij: even
            else acc[q] += 0.5 * (double)s[q] + (double)cp;
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

// f(x) at a continuous point (multilinear extension of the QUBO, reading R1):
// partial[rb][b] = sum over the rows of block rb of x_i ((Q_off x)_i + c'_i); products in fp32, sums in fp64
__global__ void __launch_bounds__(THREADS)
spmm_value(int n, int B, int rows_per_block, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
           const float* __restrict__ val2, const float* __restrict__ cprime, const float* __restrict__ x,
           double* __restrict__ partial) {
    __shared__ double red[WARPS][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool active = 4 * (blockIdx.y * 32 + lane) < B;
    const int c4 = active ? blockIdx.y * 32 + lane : B / 4 - 1;
    const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int r = warp; r < rows_per_block; r += WARPS) {
        const int row = blockIdx.x * rows_per_block + r;
        if (row >= n) break;                                 // warp-uniform
        const float4 G = gather_row(col, val2, __ldg(rowptr + row), __ldg(rowptr + row + 1), xb, 4u * (uint32_t)B, lane);
        const float4 xi = ldg4(x + (size_t)row * B + 4 * c4);
        const float cp = __ldg(cprime + row);
        acc[0] += (double)(xi.x * fmaf(0.5f, G.x, cp)); acc[1] += (double)(xi.y * fmaf(0.5f, G.y, cp));   // val2 = 2 Q_ij
        acc[2] += (double)(xi.z * fmaf(0.5f, G.z, cp)); acc[3] += (double)(xi.w * fmaf(0.5f, G.w, cp));
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) red[warp][lane][q] = acc[q];
    __syncthreads();
    if (warp == 0 && active)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            double t = red[0][lane][q];
            for (int w = 1; w < WARPS; ++w) t += red[w][lane][q];
            partial[(size_t)blockIdx.x * B + 4 * c4 + q] = t;
        }
}

template <int MODE, bool DUAL>
gda_status launch_step(gda_problem* p, int32_t B, const float* x, float* y, float* xn, const UpdParams& up,
                       const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s, int64_t* launches) {
    const int chunks = (B / 4 + 31) / 32;
    if (MODE == 0 && !DUAL && B <= 64) {                      // few restarts: several rows per warp
        int G = 1;
        while (4 * G < B) G <<= 1;
        const unsigned grid = (unsigned)((p->n + WARPS * (32 / G) - 1) / (WARPS * (32 / G)));
#define GDA_NW_CASE(GG) case GG: \
        if (up.gfun == GDA_G_QUADRATIC) spmm_step_narrow<GDA_G_QUADRATIC, GG><<<grid, THREADS, 0, s>>>(p->n, B, p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, st, t_off); \
        else spmm_step_narrow<GDA_G_ENTROPY, GG><<<grid, THREADS, 0, s>>>(p->n, B, p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, st, t_off); break;
        switch (G) { GDA_NW_CASE(1) GDA_NW_CASE(2) GDA_NW_CASE(4) GDA_NW_CASE(8) GDA_NW_CASE(16) default: break; }
#undef GDA_NW_CASE
        if (launches) ++*launches;
        GDA_CUDA_TRY(cudaGetLastError());
        return GDA_OK;
    }
    const int n_light = p->d_light_rows ? p->n_light : p->n;
    const int light_blocks = (n_light + WARPS - 1) / WARPS;
    if (n_light > 0) {
        const dim3 grid((unsigned)light_blocks, (unsigned)chunks);
#define GDA_SP_ARGS n_light, p->d_light_rows, B, p->d_rowptr, p->d_col, p->d_val2, p->d_ell, p->d_cprime, x, y, xn, up, sd, st, t_off
#define GDA_SP_CASE(E) \
        if (up.gfun == GDA_G_QUADRATIC) spmm_step_warp<GDA_G_QUADRATIC, MODE, E, DUAL><<<grid, THREADS, 0, s>>>(GDA_SP_ARGS); \
        else spmm_step_warp<GDA_G_ENTROPY, MODE, E, DUAL><<<grid, THREADS, 0, s>>>(GDA_SP_ARGS)
        if (p->d_ell) { GDA_SP_CASE(true); } else { GDA_SP_CASE(false); }
#undef GDA_SP_CASE
#undef GDA_SP_ARGS
        if (launches) ++*launches;
    }
    if (p->n_heavy > 0) {
        const unsigned grid = (unsigned)(p->n_heavy * chunks);
        if (up.gfun == GDA_G_QUADRATIC)
            spmm_step_split<GDA_G_QUADRATIC, MODE, DUAL><<<grid, THREADS, 0, s>>>(p->n_heavy, p->d_heavy_rows, B, chunks, p->d_rowptr,
                p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, sd, light_blocks, st, t_off);
        else
            spmm_step_split<GDA_G_ENTROPY, MODE, DUAL><<<grid, THREADS, 0, s>>>(p->n_heavy, p->d_heavy_rows, B, chunks, p->d_rowptr,
                p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, sd, light_blocks, st, t_off);
        if (launches) ++*launches;
    }
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

}  // namespace

int sparse_heavy_threshold() { return HEAVY_DEG; }

// shared-memory opt-in of the resident kernels on the handle's device; called at create (never inside a capture)
gda_status sparse_configure(gda_problem*) {
    GDA_CUDA_TRY(cudaFuncSetAttribute(spmm_steps_resident<GDA_G_QUADRATIC>, cudaFuncAttributeMaxDynamicSharedMemorySize, RESIDENT_SMEM));
    GDA_CUDA_TRY(cudaFuncSetAttribute(spmm_steps_resident<GDA_G_ENTROPY>, cudaFuncAttributeMaxDynamicSharedMemorySize, RESIDENT_SMEM));
    return GDA_OK;
}

gda_status sparse_step(gda_problem* p, int32_t B, const float* x, float* y, float* xn, const UpdParams& up,
                       const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s, int64_t* launches) {
    if (sd.mu) return launch_step<0, true>(p, B, x, y, xn, up, sd, st, t_off, s, launches);
    return launch_step<0, false>(p, B, x, y, xn, up, sd, st, t_off, s, launches);
}

// PDBO-s: rows of sd.gpart written per step (one per block of the warp-per-row launch, one per heavy row)
int32_t sparse_num_gparts(const gda_problem* p) {
    const int n_light = p->d_light_rows ? p->n_light : p->n;
    return (n_light + WARPS - 1) / WARPS + p->n_heavy;
}

gda_status sparse_grad(gda_problem* p, int32_t B, const float* x, float* G, cudaStream_t s) {
    UpdParams up{};
    up.gfun = GDA_G_QUADRATIC;
    return launch_step<1, false>(p, B, x, nullptr, G, up, ScalarDual{}, nullptr, 0, s, nullptr);
}

// rows per block of the scoring kernels: 64, halved down to 8 (one per warp) while the grid would leave SMs without
// two blocks (config 2: n = 800, 8 chunks -> 16 rows per block, 400 blocks)
static int score_rows(const gda_problem* p, int32_t B) {
    const long long chunks = (B / 4 + 31) / 32;
    int rows = SCORE_ROWS;
    while (rows > WARPS && ((p->n + rows - 1) / rows) * chunks < 2LL * p->num_sms) rows >>= 1;
    return rows;
}

int32_t sparse_num_partials(const gda_problem* p, int32_t B) { const int r = score_rows(p, B); return (p->n + r - 1) / r; }

gda_status sparse_score_partials(gda_problem* p, int32_t B, const float* x, void* partial, int32_t* n_part,
                                 cudaStream_t s, int64_t* launches) {
    const int chunks = (B / 4 + 31) / 32;
    dim3 grid((unsigned)sparse_num_partials(p, B), (unsigned)chunks);
    if (p->integral)
        spmm_score<true><<<grid, THREADS, 0, s>>>(p->n, B, score_rows(p, B), p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x, partial);
    else
        spmm_score<false><<<grid, THREADS, 0, s>>>(p->n, B, score_rows(p, B), p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x, partial);
    if (launches) ++*launches;
    *n_part = (int32_t)grid.x;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status sparse_value_partials(gda_problem* p, int32_t B, const float* x, double* partial, int32_t* n_part, cudaStream_t s) {
    const dim3 grid((unsigned)sparse_num_partials(p, B), (unsigned)((B / 4 + 31) / 32));
    spmm_value<<<grid, THREADS, 0, s>>>(p->n, B, score_rows(p, B), p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x, partial);
    *n_part = (int32_t)grid.x;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

// `len` steps in one launch when the state fits one block's shared memory; *done = 0 when it does not
gda_status sparse_steps_resident(gda_problem* p, int32_t B, int32_t len, const float* x_in, float* y, float* x_out,
                                 const UpdParams& up, const RunState* st, cudaStream_t s, int64_t* launches, int* done) {
    *done = 0;
    const long long total = (long long)p->n * B;
    const size_t smem = ((size_t)total * 3 + (size_t)p->n * 2 + 1 + (size_t)p->nnz * 2) * sizeof(float);   // x, x, y, c', rowptr, col, val
    if (total > RESIDENT_MAX || len <= 0 || smem > (size_t)RESIDENT_SMEM) return GDA_OK;
    if (up.gfun == GDA_G_QUADRATIC)
        spmm_steps_resident<GDA_G_QUADRATIC><<<1, RESIDENT_THREADS, smem, s>>>(p->n, B, (int)p->nnz, len, p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x_in, y, x_out, up, st);
    else
        spmm_steps_resident<GDA_G_ENTROPY><<<1, RESIDENT_THREADS, smem, s>>>(p->n, B, (int)p->nnz, len, p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x_in, y, x_out, up, st);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    *done = 1;
    return GDA_OK;
}
