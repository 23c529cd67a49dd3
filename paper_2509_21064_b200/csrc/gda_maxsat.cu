// gda_maxsat.cu -- S3 + S4 for weighted MaxSAT: per-clause literal products gathered back to variables
// through a precomputed variable-to-clause CSC, fused with the GDA update; S5 scoring by clause.
//
//   f(x) = sum_j w_j prod_{l in C_j} p_l(x),  p = 1 - x (positive literal) or x (negated)
//   G_i  = sum_{j : i in C_j} w_j s_ji prod_{l in C_j, l != i} p_l(x),  s = -1 / +1          (leave-one-out)
//
// Variable-major gather, no atomics: occurrence slot s of variable i holds coef = w_j s_ji and the kw =
// kmax-1 OTHER literals of its clause (0-padded), so the leave-one-out product is recomputed from X
// (L2-resident) instead of being stored per literal (that would add 2 x 4 x L x B bytes of HBM traffic).
// With restarts across lanes ([n][B] layout) every product is lane-local; warp shuffles only broadcast
// the slot records, which are fetched with one coalesced load per 32 slots.
#include "gda_internal.cuh"

#include <algorithm>

namespace {

constexpr int WARPS = 8;
constexpr int THREADS = WARPS * 32;
// warps per block of the step kernel: 2 -- a block's slot frees only when its slowest warp is done (config 5: 41.05 us per
// step with 8 warps, 39.75 with 4, 39.35 with 2); PDBO-s: 8, one gpart row per block of 8 variables
__host__ __device__ constexpr int step_warps(bool dual) { return dual ? WARPS : 2; }
constexpr int SCORE_CLAUSES = 128;
#ifndef GDA_MS_SLOTS_PER_BATCH
#define GDA_MS_SLOTS_PER_BATCH 2
#endif

// Slot records hold each OTHER literal encoded as  enc = var | (positive ? 0x80000000 : 0);  ENC_PAD marks padding.
// p_l(x) = off + sgn * x with (off, sgn) = (1, -1) for a positive literal and (0, +1) for a negated one.
// xb = this lane's column base (byte pointer), stride = 4*B bytes per variable.
constexpr uint32_t ENC_PAD = 0x7FFFFFFFu;
__device__ __forceinline__ float4 lit_term(uint32_t enc, const char* __restrict__ xb, uint32_t stride) {
    const uint32_t v = enc & 0x7FFFFFFFu;
    const float4 g = __ldg(reinterpret_cast<const float4*>(xb + (uint64_t)v * (uint64_t)stride));
    const float sgn = __uint_as_float((enc & 0x80000000u) | 0x3F800000u);        // -1 (positive literal) or +1 (negated)
    const float off = fmaf(sgn, -0.5f, 0.5f);                                    //  1                     or  0
    return make_float4(fmaf(sgn, g.x, off), fmaf(sgn, g.y, off), fmaf(sgn, g.z, off), fmaf(sgn, g.w, off));
}

// KW > 0: compile-time number of "other" literals (3-SAT: 2), slot records broadcast by shuffle; PAD says whether
// records may hold 0-padding (clauses shorter than kmax).  KW == 0: run-time kw, records read with broadcast loads.
// Few restarts (B <= 64): the warp's lanes form ngrp groups of 32 / ngrp lanes; a group covers all restarts and the groups
// take DIFFERENT slots of the variable at the same time (group grp: slots grp, grp + ngrp, ...) -- with one group and 3 of
// 32 lanes active at B = 12 the 13 slots of a variable are 13 dependent round trips.  The caller adds the groups' sums.
template <int KW, bool PAD>
__device__ __forceinline__ float4 gather_var(const float* __restrict__ coef, const int32_t* __restrict__ others,
                                             int kw, int start, int end, const float* __restrict__ x, int B,
                                             int c4, bool active, int lane, int grp = 0, int ngrp = 1) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (KW > 0) {
        const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
        const uint32_t stride = 4u * (uint32_t)B;
        for (int base = start; base < end; base += 32) {
            const int s = base + lane;
            const float my_coef = (s < end) ? __ldg(coef + s) : 0.0f;
            int my_o[KW > 0 ? KW : 1];
#pragma unroll
            for (int q = 0; q < KW; ++q) my_o[q] = (s < end) ? __ldg(others + (size_t)s * KW + q) : (int)ENC_PAD;
            const int cnt = min(32, end - base);
            constexpr int U = GDA_MS_SLOTS_PER_BATCH;             // slots per batch: U*KW independent 512 B gathers in flight
            for (int u0 = 0; u0 < cnt; u0 += U * ngrp) {
                float cf[U]; int l[U][KW > 0 ? KW : 1]; float4 t[U][KW > 0 ? KW : 1];
#pragma unroll
                for (int a = 0; a < U; ++a) {                     // past the end: re-read the last slot with coefficient 0
                    const int idx = u0 + a * ngrp + grp;
                    const int src = min(idx, cnt - 1);
                    cf[a] = __shfl_sync(0xffffffffu, my_coef, src);
#pragma unroll
                    for (int q = 0; q < KW; ++q) l[a][q] = __shfl_sync(0xffffffffu, my_o[q], src);
                    if (idx >= cnt) cf[a] = 0.0f;
                }
                if (!active) continue;
#pragma unroll
                for (int a = 0; a < U; ++a)
#pragma unroll
                    for (int q = 0; q < KW; ++q) {
                        if (PAD && (uint32_t)l[a][q] == ENC_PAD) { t[a][q] = make_float4(1.f, 1.f, 1.f, 1.f); continue; }
                        t[a][q] = lit_term((uint32_t)l[a][q], xb, stride);
                    }
#pragma unroll
                for (int a = 0; a < U; ++a) {                     // acc += cf * t0 * t1 * ... (last factor fused into the add)
                    float4 prod = make_float4(cf[a] * t[a][0].x, cf[a] * t[a][0].y, cf[a] * t[a][0].z, cf[a] * t[a][0].w);
#pragma unroll
                    for (int q = 1; q + 1 < KW; ++q) { prod.x *= t[a][q].x; prod.y *= t[a][q].y; prod.z *= t[a][q].z; prod.w *= t[a][q].w; }
                    if (KW > 1) {
                        acc.x = fmaf(prod.x, t[a][KW - 1].x, acc.x); acc.y = fmaf(prod.y, t[a][KW - 1].y, acc.y);
                        acc.z = fmaf(prod.z, t[a][KW - 1].z, acc.z); acc.w = fmaf(prod.w, t[a][KW - 1].w, acc.w);
                    } else {
                        acc.x += prod.x; acc.y += prod.y; acc.z += prod.z; acc.w += prod.w;
                    }
                }
            }
        }
    } else {
        if (!active) return acc;
        const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
        const uint32_t stride = 4u * (uint32_t)B;
        for (int s = start; s < end; ++s) {
            const float cf = __ldg(coef + s);
            float4 prod = make_float4(cf, cf, cf, cf);
            for (int q = 0; q < kw; ++q) {
                const uint32_t l = (uint32_t)__ldg(others + (size_t)s * kw + q);
                if (l == ENC_PAD) break;
                const float4 t = lit_term(l, xb, stride);
                prod.x *= t.x; prod.y *= t.y; prod.z *= t.z; prod.w *= t.w;
            }
            acc.x += prod.x; acc.y += prod.y; acc.z += prod.z; acc.w += prod.w;
        }
    }
    return acc;
}

// warp-per-(variable, 128-restart chunk): blockIdx.y = chunk, the block's 8 warps take 8 consecutive variables.
// MODE 0: fused step; MODE 1: write G only.  DUAL (PDBO-s, MODE 0): one multiplier per restart (sd.mu),
// y untouched, the block's sum of g(x_i^t) goes to sd.gpart[blockIdx.x].
// NARROW (B <= 64, step only, KW > 0): lanes_per_group = the power of two >= B / 4 lanes cover the restarts, the warp's
// 32 / lanes_per_group groups share the slots of the variable (gather_var) and their sums are added by a butterfly.
template <int GFUN, int MODE, int KW, bool PAD, bool DUAL, bool NARROW = false>
__global__ void __launch_bounds__(32 * step_warps(DUAL))
maxsat_step_kernel(int n, int B, const int32_t* __restrict__ vptr, const float* __restrict__ coef,
                   const int32_t* __restrict__ others, int kw, const float* __restrict__ x,
                   float* __restrict__ y, float* __restrict__ xn, UpdParams up, ScalarDual sd,
                   const RunState* __restrict__ st, uint32_t t_off, int lanes_per_group = 32) {
    constexpr int SW = step_warps(DUAL);
    __shared__ float4 gred[DUAL ? SW : 1][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = NARROW ? lane / lanes_per_group : 0, ngrp = NARROW ? 32 / lanes_per_group : 1;
    const int c4 = NARROW ? lane % lanes_per_group : blockIdx.y * 32 + lane;
    const bool active = 4 * c4 < B;
    float4 gs = make_float4(0.f, 0.f, 0.f, 0.f), mu = gs;
    if (DUAL) mu = ldg4(sd.mu + 4 * (active ? c4 : B / 4 - 1));
    const int var = blockIdx.x * SW + warp;
    if (var < n) {                                           // warp-uniform
        const int start = __ldg(vptr + var), end = __ldg(vptr + var + 1);
        float4 G = gather_var<KW, PAD>(coef, others, kw, start, end, x, B, c4, active, lane, grp, ngrp);
        if (NARROW) {
            for (int o = lanes_per_group; o < 32; o <<= 1) {  // the groups' sums, in a fixed order
                G.x += __shfl_xor_sync(0xffffffffu, G.x, o); G.y += __shfl_xor_sync(0xffffffffu, G.y, o);
                G.z += __shfl_xor_sync(0xffffffffu, G.z, o); G.w += __shfl_xor_sync(0xffffffffu, G.w, o);
            }
        }
        if (active && grp == 0) {
            const size_t off = (size_t)var * B + 4 * c4;
            if (MODE == 1) {
                *reinterpret_cast<float4*>(xn + off) = G;
            } else {
                const uint32_t t = (st ? st->t : 0u) + t_off;
                const float4 xv = ldg4(x + off);
                const float4 yv = DUAL ? mu : *reinterpret_cast<const float4*>(y + off);
                float4 xo, yo;
                gda_update4<GFUN>(xv, yv, G, up, t, (uint32_t)var, 4u * (uint32_t)c4, xo, yo);
                *reinterpret_cast<float4*>(xn + off) = xo;
                if (DUAL) gs = make_float4(gda_g<GFUN>(xv.x, up), gda_g<GFUN>(xv.y, up), gda_g<GFUN>(xv.z, up), gda_g<GFUN>(xv.w, up));
                else *reinterpret_cast<float4*>(y + off) = yo;
            }
        }
    }
    if (DUAL) scalar_dual_block_sum<SW>(gs, gred, warp, lane, active, sd.gpart + (size_t)blockIdx.x * B + 4 * c4);
}

// S5: partial[cb][b] = sum over the clauses of block cb of w_j [every literal of C_j false under x_hat]
template <bool INTEGRAL>
__global__ void __launch_bounds__(THREADS)
maxsat_score(int m, int B, int clauses_per_block, const int32_t* __restrict__ cptr, const int32_t* __restrict__ lit,
             const float* __restrict__ w, const float* __restrict__ x, void* __restrict__ partial) {
    using acc_t = typename std::conditional<INTEGRAL, long long, double>::type;
    __shared__ acc_t red[WARPS][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c4 = blockIdx.y * 32 + lane;
    const bool active = 4 * c4 < B;
    acc_t acc[4] = {0, 0, 0, 0};
    if (active) {
        for (int r = warp; r < clauses_per_block; r += WARPS) {
            const int j = blockIdx.x * clauses_per_block + r;
            if (j >= m) break;
            bool unsat[4] = {true, true, true, true};
            for (int a = __ldg(cptr + j); a < __ldg(cptr + j + 1); ++a) {
                const int l = __ldg(lit + a);
                const int v = (l > 0 ? l : -l) - 1;
                const float4 g = ldg4(x + (size_t)v * B + 4 * c4);
                const bool h[4] = {g.x > 0.5f, g.y > 0.5f, g.z > 0.5f, g.w > 0.5f};
#pragma unroll
                for (int q = 0; q < 4; ++q) unsat[q] = unsat[q] && (l > 0 ? !h[q] : h[q]);   // literal false
            }
            const float wj = __ldg(w + j);
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (unsat[q]) acc[q] += INTEGRAL ? (acc_t)__float2int_rn(wj) : (acc_t)wj;
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
            for (int k = 1; k < WARPS; ++k) t += red[k][lane][q];
            out[q] = t;
        }
    }
}

// f(x) at a continuous point: partial[cb][b] = sum over the clauses of block cb of w_j prod_{l in C_j} p_l(x)
// (PAPER.md:196); products in fp32, sums in fp64
__global__ void __launch_bounds__(THREADS)
maxsat_value(int m, int B, int clauses_per_block, const int32_t* __restrict__ cptr, const int32_t* __restrict__ lit,
             const float* __restrict__ w, const float* __restrict__ x, double* __restrict__ partial) {
    __shared__ double red[WARPS][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c4 = blockIdx.y * 32 + lane;
    const bool active = 4 * c4 < B;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    if (active)
        for (int r = warp; r < clauses_per_block; r += WARPS) {
            const int j = blockIdx.x * clauses_per_block + r;
            if (j >= m) break;
            const float wj = __ldg(w + j);
            float4 prod = make_float4(wj, wj, wj, wj);
            for (int a = __ldg(cptr + j); a < __ldg(cptr + j + 1); ++a) {
                const int l = __ldg(lit + a);
                const float4 g = ldg4(x + (size_t)((l > 0 ? l : -l) - 1) * B + 4 * c4);
                if (l > 0) { prod.x *= 1.0f - g.x; prod.y *= 1.0f - g.y; prod.z *= 1.0f - g.z; prod.w *= 1.0f - g.w; }
                else { prod.x *= g.x; prod.y *= g.y; prod.z *= g.z; prod.w *= g.w; }
            }
            acc[0] += (double)prod.x; acc[1] += (double)prod.y; acc[2] += (double)prod.z; acc[3] += (double)prod.w;
        }
#pragma unroll
    for (int q = 0; q < 4; ++q) red[warp][lane][q] = acc[q];
    __syncthreads();
    if (warp == 0 && active)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            double t = red[0][lane][q];
            for (int k = 1; k < WARPS; ++k) t += red[k][lane][q];
            partial[(size_t)blockIdx.x * B + 4 * c4 + q] = t;
        }
}

template <int GFUN, int MODE, bool DUAL>
void launch_kw(gda_problem* p, int32_t B, dim3 grid, const float* x, float* y, float* xn,
               const UpdParams& up, const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s) {
#define GDA_MS_ARGS p->n, B, p->d_vptr, p->d_coef, p->d_others, p->kw, x, y, xn, up, sd, st, t_off
#define GDA_MS_CASE(K) \
        case K: if (narrow) { if (pad) maxsat_step_kernel<GFUN, 0, K, true, false, true><<<grid, 32 * step_warps(false), 0, s>>>(GDA_MS_ARGS, lanes); \
                              else maxsat_step_kernel<GFUN, 0, K, false, false, true><<<grid, 32 * step_warps(false), 0, s>>>(GDA_MS_ARGS, lanes); } \
                else if (pad) maxsat_step_kernel<GFUN, MODE, K, true, DUAL><<<grid, 32 * step_warps(DUAL), 0, s>>>(GDA_MS_ARGS); \
                else maxsat_step_kernel<GFUN, MODE, K, false, DUAL><<<grid, 32 * step_warps(DUAL), 0, s>>>(GDA_MS_ARGS); break;
    // records hold ENC_PAD when clauses are shorter than kmax -- and ALWAYS when kmax == 1 (kw is then 1 with no other literal)
    const bool pad = p->kmin != p->kmax || p->kmax == 1;
    // few restarts: slot groups (gather_var); B <= 64 is one 128-restart chunk, so grid.y == 1
    const bool narrow = MODE == 0 && !DUAL && B <= 64 && p->kw <= 4 && p->opt_maxsat_narrow;   // GDA_OPT_MAXSAT_NARROW
    int lanes = 1;
    while (4 * lanes < B) lanes <<= 1;
    switch (p->kw) {
        GDA_MS_CASE(1) GDA_MS_CASE(2) GDA_MS_CASE(3) GDA_MS_CASE(4)
        default: maxsat_step_kernel<GFUN, MODE, 0, true, DUAL><<<grid, 32 * step_warps(DUAL), 0, s>>>(GDA_MS_ARGS); break;
    }
#undef GDA_MS_CASE
#undef GDA_MS_ARGS
}

template <int MODE, bool DUAL>
gda_status launch_step(gda_problem* p, int32_t B, const float* x, float* y, float* xn, const UpdParams& up,
                       const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s, int64_t* launches) {
    const int groups = (p->n + step_warps(DUAL) - 1) / step_warps(DUAL), chunks = (B / 4 + 31) / 32;
    const dim3 grid((unsigned)groups, (unsigned)chunks);
    if (up.gfun == GDA_G_QUADRATIC) launch_kw<GDA_G_QUADRATIC, MODE, DUAL>(p, B, grid, x, y, xn, up, sd, st, t_off, s);
    else launch_kw<GDA_G_ENTROPY, MODE, DUAL>(p, B, grid, x, y, xn, up, sd, st, t_off, s);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

}  // namespace

gda_status maxsat_step(gda_problem* p, int32_t B, const float* x, float* y, float* xn, const UpdParams& up,
                       const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s, int64_t* launches) {
    if (sd.mu) return launch_step<0, true>(p, B, x, y, xn, up, sd, st, t_off, s, launches);
    return launch_step<0, false>(p, B, x, y, xn, up, sd, st, t_off, s, launches);
}

int32_t maxsat_num_gparts(const gda_problem* p) { return (p->n + WARPS - 1) / WARPS; }

gda_status maxsat_grad(gda_problem* p, int32_t B, const float* x, float* G, cudaStream_t s) {
    UpdParams up{};
    up.gfun = GDA_G_QUADRATIC;
    return launch_step<1, false>(p, B, x, nullptr, G, up, ScalarDual{}, nullptr, 0, s, nullptr);
}

// clauses per block of the scoring kernels: at most SCORE_CLAUSES, fewer when that grid would leave the machine idle -- a warp
// walks its clauses one after the other (config 5 at B = 10: 333 blocks, 16 clauses per warp, 25 us per evaluation)
static int score_clauses(const gda_problem* p, int32_t B) {
    const int64_t chunks = (B / 4 + 31) / 32;
    const int64_t want = ((int64_t)p->m * chunks / ((int64_t)p->num_sms * 8) + 7) / 8 * 8;
    return (int)std::min<int64_t>(SCORE_CLAUSES, std::max<int64_t>(8, want));
}
int32_t maxsat_num_partials(const gda_problem* p, int32_t B) { const int c = score_clauses(p, B); return (p->m + c - 1) / c; }

gda_status maxsat_score_partials(gda_problem* p, int32_t B, const float* x, void* partial, int32_t* n_part,
                                 cudaStream_t s, int64_t* launches) {
    const int chunks = (B / 4 + 31) / 32;
    dim3 grid((unsigned)maxsat_num_partials(p, B), (unsigned)chunks);
    if (p->integral)
        maxsat_score<true><<<grid, THREADS, 0, s>>>(p->m, B, score_clauses(p, B), p->d_cptr, p->d_lit, p->d_w, x, partial);
    else
        maxsat_score<false><<<grid, THREADS, 0, s>>>(p->m, B, score_clauses(p, B), p->d_cptr, p->d_lit, p->d_w, x, partial);
    if (launches) ++*launches;
    *n_part = (int32_t)grid.x;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status maxsat_value_partials(gda_problem* p, int32_t B, const float* x, double* partial, int32_t* n_part, cudaStream_t s) {
    const dim3 grid((unsigned)maxsat_num_partials(p, B), (unsigned)((B / 4 + 31) / 32));
    maxsat_value<<<grid, THREADS, 0, s>>>(p->m, B, score_clauses(p, B), p->d_cptr, p->d_lit, p->d_w, x, partial);
    *n_part = (int32_t)grid.x;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}
