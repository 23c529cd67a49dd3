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

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <math_constants.h>
#define CUDART_INF_SLAB CUDART_INF

namespace {

constexpr int WARPS = 8;
constexpr int THREADS = WARPS * 32;
// warps per block of spmm_step_warp: 4 (12 blocks per SM) -- a block's slot is free only when its slowest warp is done, and
// with 4 warps less of the SM waits (config 3: 14.9 -> 14.4 us per step, B = 1024: 66.6 -> 63.9 us); PDBO-s keeps 8: every
// block ends in a reduction and a set of atomics, and twice the blocks cost more than they gain (19.1 -> 21.7 us)
// Config 2's graph (n = 800, degree 48) through the streaming kernels, us per step: B = 100 8.66 with a warp per row, 4.38 with
// the rows split; B = 256 8.72 / 6.58; B = 512 9.10 / 11.21; B = 1024 12.08 / 20.37 (the slab kernel: 8.4 at any B).
static bool split_all_rows(const gda_problem* p, int32_t B) {
    if (p->opt_split_all >= 0) return p->opt_split_all == 1;      // GDA_OPT_SPLIT_ALL_ROWS
    const int64_t chunks = (B / 4 + 31) / 32;
    return B > 32 && (int64_t)p->n * chunks < (int64_t)p->num_sms * 12 && p->nnz >= 16 * (int64_t)p->n;   // B <= 32: the narrow kernel splits rows itself
}
// narrow kernel (B <= 64): lane groups per row, as many as give every group about two batches of four entries of an average row
static int narrow_split_log2(const gda_problem* p, int32_t B) {
    if (!p->opt_narrow_split) return 0;                           // GDA_OPT_NARROW_SPLIT
    int G = 1, split_log2 = 0;
    while (4 * G < B) G <<= 1;
    while ((G << (split_log2 + 1)) <= 32 && (8 << (split_log2 + 1)) <= p->nnz / std::max(p->n, 1)) ++split_log2;
    return split_log2;
}
__host__ __device__ constexpr int warp_kernel_warps(bool dual) { return dual ? 8 : 4; }
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
// not touched, and g of the NEW iterate x^{t+1} is returned in gs (0 for lanes past a ragged B): the sum the multiplier
// update of the NEXT iteration needs (ScalarDual in gda_internal.cuh).
template <int GFUN, bool DUAL>
__device__ __forceinline__ void update_store(int row, int c4, int B, bool active, float4 G, const float* __restrict__ x,
                                             float* __restrict__ y, float* __restrict__ xn,
                                             const UpdParams& up, uint32_t t, float4 mu, float4& gs) {
    // byte offset of (row, c4) as ONE 32 x 32 -> 64-bit multiply-add per array (n * B < 2^30 elements is checked by
    // gda_run): the generic 64-bit index arithmetic costs a dozen instructions and a register pair more
    const uint64_t off = (uint64_t)(uint32_t)row * (uint64_t)(4u * (uint32_t)B) + (uint64_t)(16u * (uint32_t)c4);
    const float4 xv = __ldg(reinterpret_cast<const float4*>(reinterpret_cast<const char*>(x) + off));
    float4* yp = reinterpret_cast<float4*>(reinterpret_cast<char*>(y) + off);
    const float4 yv = DUAL ? mu : *yp;
    float4 xo, yo;
    gda_update4<GFUN>(xv, yv, G, up, t, (uint32_t)row, 4u * (uint32_t)c4, xo, yo);
    if (!active) return;
    *reinterpret_cast<float4*>(reinterpret_cast<char*>(xn) + off) = xo;
    if (DUAL) gs = make_float4(gda_g<GFUN>(xo.x, up), gda_g<GFUN>(xo.y, up), gda_g<GFUN>(xo.z, up), gda_g<GFUN>(xo.w, up));   // g of x^{t+1}: S^{t+1}
    else *yp = yo;
}

// warp-per-(row, 128-restart chunk): blockIdx.y = chunk, the block's 8 warps take 8 consecutive rows.
// MODE 0: fused step, MODE 1: write G only (gda_grad).
// ELL: rows of degree <= 8 come as one packed 64-byte record (8 columns, 8 values; gda_api.cu) fetched with a single
// coalesced load, which removes the rowptr -> (col, val) hop from the dependent chain of a row; a record whose word 0
// is -1 sends the row through its CSR entries.  40 registers (6 blocks per SM).  Measured on config 3 (profiles/):
// 17.3 us per step before, 16.3 us with the lean gather loop, 14.8 us with the records and 6 blocks per SM;
// prefetching the row's own x, y lines into L1 up front was slower (15.1 us) and is not done.
// DUAL (PDBO-s, MODE 0 only): the multiplier is one number per restart (sd.mu), y is not read or written, and the
// block's sum of g over the values it writes goes through scalar_dual_finish (fixed-point integer reductions); block 0 of
// every chunk also closes the multiplier update of this iteration from the sums the previous kernel left (scalar_dual_advance).
template <int GFUN, int MODE, bool ELL, bool DUAL, bool PF>
__global__ void __launch_bounds__(32 * warp_kernel_warps(DUAL), 6 * 8 / warp_kernel_warps(DUAL))
spmm_step_warp(int n_rows, const int32_t* __restrict__ row_list, int B,
               const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
               const float* __restrict__ val2, const int32_t* __restrict__ ell, const float* __restrict__ cprime,
               const float* __restrict__ x, float* __restrict__ y, float* __restrict__ xn,
               UpdParams up, ScalarDual sd, const RunState* __restrict__ st, uint32_t t_off) {
    constexpr int WW = warp_kernel_warps(DUAL);
    __shared__ float4 gred[DUAL ? WW : 1][32];
    __shared__ long long adv[DUAL ? WW : 1][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ridx = blockIdx.x * WW + warp;
    const bool active = 4 * (blockIdx.y * 32 + lane) < B;
    const int c4 = active ? blockIdx.y * 32 + lane : B / 4 - 1;      // ragged B: idle lanes recompute the last float4
    if (DUAL) {
        float4 gs = make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 mu = ldg4(sd.mu + 4 * c4);
        if (sd.advance && blockIdx.x == 0) scalar_dual_advance<WW>(adv, warp, lane, active, c4, sd);   // block-uniform: mu^{t+1} for this chunk's restarts
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
        scalar_dual_finish<WW>(gs, gred, warp, lane, active, c4, blockIdx.x, sd);
        return;
    }
    if (ridx >= n_rows) return;                              // warp-uniform
    const int row = row_list ? __ldg(row_list + ridx) : ridx;
    const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
    const uint32_t stride = 4u * (uint32_t)B;
    // HBM-streaming case (the state does not fit L2: PF): start the row's own x, y lines towards L2 now, so
    // that the DRAM latency hides behind the gather chain (config 3's graph at B = 1024: 73.2 -> 67.6 us per step; with
    // an L2-resident state the extra instructions cost 2.5 %, hence the switch)
    if (MODE == 0 && PF && (lane & 7) == 0) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(x + (size_t)row * B + 4 * c4));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(y + (size_t)row * B + 4 * c4));
    }
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
constexpr int NARROW_WARPS = 4;      // per block (MIS n = 5e4, d = 100, B = 12: 46.6 us per step with 8, 42.5 with 4 or 2, 46.1 with 1)
// Long rows with few restarts (MIS d = 100 at B = 10: 100 entries per row, 1 250 warps in all at n = 10^4) are split further:
// S = 2^split_log2 lane groups per row take the row's batches of four entries in turn (group s: batches s, s + S, ...) and add
// their sums by a butterfly; a warp then holds 32 / (G S) rows.
template <int GFUN, int G>
__global__ void __launch_bounds__(32 * NARROW_WARPS)
spmm_step_narrow(int n, int B, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                 const float* __restrict__ val2, const float* __restrict__ cprime, const float* __restrict__ x,
                 float* __restrict__ y, float* __restrict__ xn, UpdParams up, const RunState* __restrict__ st, uint32_t t_off,
                 int split_log2) {
    const int S = 1 << split_log2, R = 32 / (G * S);         // lane groups per row, rows per warp
    const int lane = threadIdx.x & 31;
    const int row_raw = (blockIdx.x * NARROW_WARPS + (threadIdx.x >> 5)) * R + lane / (G * S);
    const int cl = lane % G, sg = (lane / G) & (S - 1);
    const bool active = row_raw < n && 4 * cl < B && sg == 0;
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
    for (int a = 4 * sg; a < maxdeg; a += 4 * S) {
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
    for (int o = G; o < G * S; o <<= 1) {                    // the row's lane groups, in a fixed order
        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
        acc.z += __shfl_xor_sync(0xffffffffu, acc.z, o); acc.w += __shfl_xor_sync(0xffffffffu, acc.w, o);
    }
    const float cp = __ldg(cprime + row);
    acc.x += cp; acc.y += cp; acc.z += cp; acc.w += cp;
    float4 unused;
    update_store<GFUN, false>(row, c4, B, active, acc, x, y, xn, up, (st ? st->t : 0u) + t_off, make_float4(0.f, 0.f, 0.f, 0.f), unused);
}

// row-split: one block per (row, chunk); the 8 warps take interleaved slices of `slice` entries of the row (32 for the rows
// above HEAVY_DEG).  row_list == NULL: every row -- used with slices of 8 when the whole launch would otherwise be a few warps
// per SM that each walk a long row (n = 800, degree 48 at B = 100, the paper's batch size on the 800-node Gset graphs: 800
// warps in all; 8.7 -> see launch_step).  DUAL: as above.
template <int GFUN, int MODE, bool DUAL>
__global__ void __launch_bounds__(THREADS)
spmm_step_split(int n_rows, const int32_t* __restrict__ row_list, int B, int chunks,
                const int32_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                const float* __restrict__ val2, const float* __restrict__ cprime,
                const float* __restrict__ x, float* __restrict__ y, float* __restrict__ xn,
                UpdParams up, ScalarDual sd, const RunState* __restrict__ st, uint32_t t_off, int slice) {
    __shared__ float4 red[WARPS][32];
    __shared__ long long adv[DUAL ? WARPS : 1][32][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ridx = blockIdx.x / chunks, chunk = blockIdx.x % chunks;
    const int row = row_list ? __ldg(row_list + ridx) : ridx;
    const bool active = 4 * (chunk * 32 + lane) < B;
    const int c4 = active ? chunk * 32 + lane : B / 4 - 1;
    const char* xb = reinterpret_cast<const char*>(x + 4 * c4);
    const int start = __ldg(rowptr + row), end = __ldg(rowptr + row + 1);
    if (DUAL && sd.advance && ridx == 0) scalar_dual_advance<WARPS>(adv, warp, lane, active, c4, sd);   // block-uniform: mu^{t+1} for this chunk's restarts
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int base = start + slice * warp; base < end; base += slice * WARPS) {
        const float4 part = gather_row(col, val2, base, min(base + slice, end), xb, 4u * (uint32_t)B, lane);
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
    if (DUAL) scalar_dual_commit(gs, active, c4, (unsigned)ridx, sd);
}

// ---- slab variant for small n: a whole chunk of steps AND its evaluation in one launch ---------------------------------
// Restarts are independent, so a CTA that owns a slab of SLAB_S = 8 restarts for ALL n rows needs nobody
// else: x (double-buffered: the update is simultaneous, Eq. 6), y and c' live in shared memory for the whole chunk
// (12 B x n x 8 per CTA: n <= 2300), the steps are separated by __syncthreads(), and global memory sees the state only at
// the chunk's two ends.  The gathers -- what bounds config 2 (n = 800, degree 48: 157 MB per step out of L2 at 12 us) --
// become shared-memory reads: floor = nnz x B x 4 B / (SMs x 128 B/clk), 5 us per step for config 2.
//
// Work split: lane = (row r of a group of 16 rows, quad q of the slab's 8 restarts); every lane walks ITS OWN row, so
// there is no reduction across lanes.  The structure is a sliced ELL built at create (gda_api.cu): rows sorted by degree
// and dealt to groups of 16; slot k of a group holds one (column byte offset, 2 Q_ij) pair per row, 128 contiguous
// bytes, so the warp's fetch of slot k is ONE coalesced line (two lanes per address).  A gather is an LDS.128: the
// hardware serves 8 lanes = 4 rows x 32 B per pass, conflict-free iff the 4 columns differ mod 4 -- the entries of
// every 4 rows that share a pass are therefore ordered at create such that they do (zero-valued padding where the
// greedy matching cannot; a few per cent).
//
// The evaluation (S5, S6's per-restart part) is fused: the CTA scores its 8 restarts exactly (integers for integral
// instances, fixed summation order otherwise), updates best_obj / improved, commits x_hat of improved restarts to x_bin
// and takes part in the same last-block ticket as finalize_kernel for the trace and the run state.
constexpr int SLAB_S = 8, SLAB_ROWS = 16, SLAB_MAX_THREADS = 1024;
constexpr int SLAB_SMEM_LIMIT = 226 * 1024;                  // dynamic shared memory of a CTA (the kernel also has a few static bytes)

struct SlabArgs {
    int n, B, len, n_groups, groups_per_warp, n_pass;   // B: restarts (row stride) including padding restarts
    int B_eval;                      // restarts that count: the evaluation skips the padding restarts b >= B_eval
    const int2* ent;                 // general: [slot][16 rows] (col * 32 bytes, bits of val2)
    const uint2* ent16;              // compact: [pass][16 rows] four 16-bit entries: bit 15 = sign of val2, bits 0..11 = column
    uint32_t cbits;                  // compact: bits of |val2|, the one magnitude all entries share
    const int32_t* goff;             // [n_groups + 1] first slot of a group (lengths are multiples of 4)
    const int32_t* grow;             // [n_groups * 16] row index, -1 = no row
    const float* cprime;
    const float* x_in; float* x_out; // [n][B]: x^t is read from x_in at the start, x^{t+len} written to x_out at the end
    float* y;                        // [n][B], in place (a CTA touches nothing outside its slab, so x_in may equal x_out)
    const float* mu_in; float* mu_out;   // PDBO-s (DUAL): [B] multipliers at the chunk's start / end; y is not touched
    UpdParams up;
    RunState* st;
    double* best_obj; int32_t* improved; uint8_t* x_bin; double* block_min;
    double* trace_best; uint64_t* trace_ns; int trace_cap;
};

__device__ __forceinline__ uint64_t slab_globaltimer_ns() {
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// One pass = 4 slots of this lane's row: byte offsets of the 4 gathered rows of x and their values.
struct SlabPass { int off[4]; float val[4]; };

// COMPACT (every non-zero |2 Q_ij| is the same number: unit, +-1 or constant weights -- Max-Cut on the paper's graphs,
// MIS): 2 bytes per entry, the whole structure copied into shared memory once per chunk, so a step reads nothing but
// shared memory.  Otherwise: 8 bytes per entry from global memory (L2), fetched one pass ahead.
template <bool COMPACT>
__device__ __forceinline__ SlabPass slab_fetch(const SlabArgs& a, const uint2* __restrict__ cst, int pass, int r) {
    SlabPass p;
    if (COMPACT) {
        const uint2 w = cst[pass * SLAB_ROWS + r];
        const uint32_t e[4] = {w.x & 0xFFFFu, w.x >> 16, w.y & 0xFFFFu, w.y >> 16};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            p.off[u] = (int)((e[u] & 0xFFFu) << 5);
            p.val[u] = __uint_as_float(a.cbits ^ ((e[u] & 0x8000u) << 16));
        }
    } else {
        const int2* ep = a.ent + (size_t)pass * 4 * SLAB_ROWS + r;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int2 e = __ldg(ep + u * SLAB_ROWS);
            p.off[u] = e.x;
            p.val[u] = __int_as_float(e.y);
        }
    }
    return p;
}

// groups are sorted by falling length; warp w takes groups w, 2W-1-w, 2W+w, ... (serpentine), so that every warp gets
// long and short ones and the per-step barrier does not wait for the warp with the longest rows
__device__ __forceinline__ int slab_group(int i, int warp, int warps) { return (i & 1) ? i * warps + (warps - 1 - warp) : i * warps + warp; }

// DUAL (PDBO-s, reading R14): one multiplier per restart instead of y.  The CTA holds ALL rows of its restarts, so the sum of
// g(x_i^t) over the variables is a reduction inside the CTA -- lanes of a warp by a fixed butterfly, the warps in index order --
// and the multiplier's update costs one more barrier per step: no atomics, no second kernel, deterministic.
template <int GFUN, bool INTEGRAL, bool COMPACT, bool DUAL>
__global__ void __launch_bounds__(SLAB_MAX_THREADS, 1)
spmm_chunk_slab(const SlabArgs a) {
    using acc_t = typename std::conditional<INTEGRAL, long long, double>::type;
    extern __shared__ float4 slab_smem[];
    const int nrow = a.n + (COMPACT ? 4 : 0);                 // compact: four rows of zeros, what padding entries gather
    float* xa = reinterpret_cast<float*>(slab_smem);          // x^t  [nrow][8]
    float* xb = xa + (size_t)nrow * SLAB_S;                   // x^{t+1}
    float* ys = xb + (size_t)nrow * SLAB_S;                   // y [n][8]
    float* cps = ys + (size_t)a.n * SLAB_S;                   // c' [n]
    acc_t* red = reinterpret_cast<acc_t*>(cps + ((a.n + 3) & ~3));   // [warps][8] per-warp objective sums
    uint2* cst = reinterpret_cast<uint2*>(red + (blockDim.x >> 5) * SLAB_S);   // compact structure [n_pass][16]
    __shared__ int s_imp[SLAB_S];
    __shared__ unsigned s_last;
    __shared__ __align__(16) float s_mu[SLAB_S];                            // DUAL: this step's multipliers of the slab's restarts
    float (*s_gred)[SLAB_S] = reinterpret_cast<float (*)[SLAB_S]>(red);   // DUAL: the warps' sums of g(x_i^t) (red is free until the evaluation)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    const int r = lane >> 1, q = lane & 1;
    const int b0 = blockIdx.x * SLAB_S;                       // first restart of the slab

    // ---- load the slab (32 bytes per row and array; a ragged B, a multiple of 4, may lack the slab's second quad) ----
    for (int e = threadIdx.x; e < a.n * 2; e += blockDim.x) {
        const int row = e >> 1, qq = e & 1;
        float4 xv = make_float4(0.f, 0.f, 0.f, 0.f), yv = xv;
        if (b0 + 4 * qq < a.B) {
            const size_t off = (size_t)row * a.B + b0 + 4 * qq;
            xv = __ldcg(reinterpret_cast<const float4*>(a.x_in + off));       // not ld.global.nc: this kernel writes x (x_out may alias
            if (!DUAL) yv = __ldcg(reinterpret_cast<const float4*>(a.y + off));   // x_in), y and mu back, so they are not read-only for it
        }
        reinterpret_cast<float4*>(xa)[e] = xv;
        if (!DUAL) reinterpret_cast<float4*>(ys)[e] = yv;
    }
    if (DUAL && threadIdx.x < SLAB_S) s_mu[threadIdx.x] = b0 + (int)threadIdx.x < a.B ? __ldcg(a.mu_in + b0 + threadIdx.x) : 0.0f;
    for (int e = threadIdx.x; e < a.n; e += blockDim.x) cps[e] = __ldg(a.cprime + e);
    if (COMPACT) {
        for (int e = threadIdx.x; e < a.n_pass * SLAB_ROWS; e += blockDim.x) cst[e] = __ldg(a.ent16 + e);
        if (threadIdx.x < 8) {                                // the zero rows, in both buffers
            reinterpret_cast<float4*>(xa)[a.n * 2 + threadIdx.x] = make_float4(0.f, 0.f, 0.f, 0.f);
            reinterpret_cast<float4*>(xb)[a.n * 2 + threadIdx.x] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    __syncthreads();

    const uint32_t t0 = a.st->t;
    const char* xq = reinterpret_cast<const char*>(xa) + 16 * q;        // + column byte offset = this lane's float4 of row col

    // ---- len GDA steps, state on chip ----
    for (int k = 0; k < a.len; ++k) {
        float4 gs = make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 mu4 = DUAL ? *reinterpret_cast<const float4*>(s_mu + 4 * q) : gs;
        for (int i = 0; i < a.groups_per_warp; ++i) {
            const int g = slab_group(i, warp, warps);
            if (g >= a.n_groups) break;
            const int p0 = __ldg(a.goff + g) >> 2, p1 = __ldg(a.goff + g + 1) >> 2;
            const int row = __ldg(a.grow + g * SLAB_ROWS + r);
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
            // the structure of the NEXT pass is fetched before this pass's gathers, so that its latency hides behind them
            SlabPass cur = slab_fetch<COMPACT>(a, cst, min(p0, a.n_pass - 1), r), nxt;
#pragma unroll 1
            for (int ps = p0; ps < p1; ++ps) {
                nxt = slab_fetch<COMPACT>(a, cst, min(ps + 1, a.n_pass - 1), r);
                float4 gv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) gv[u] = *reinterpret_cast<const float4*>(xq + cur.off[u]);
#pragma unroll
                for (int u = 0; u < 4; ++u) fma4(acc, cur.val[u], gv[u]);
                cur = nxt;
            }
            if (row >= 0) {
                const float cp = cps[row];
                acc.x += cp; acc.y += cp; acc.z += cp; acc.w += cp;
                const int idx = row * 2 + q;
                const float4 xv = reinterpret_cast<const float4*>(xa)[idx];
                const float4 yv = DUAL ? mu4 : reinterpret_cast<const float4*>(ys)[idx];
                float4 xo, yo;
                gda_update4<GFUN>(xv, yv, acc, a.up, t0 + (uint32_t)k, (uint32_t)row, (uint32_t)(b0 + 4 * q), xo, yo);
                reinterpret_cast<float4*>(xb)[idx] = xo;
                if (DUAL) {
                    gs.x += gda_g<GFUN>(xv.x, a.up); gs.y += gda_g<GFUN>(xv.y, a.up);
                    gs.z += gda_g<GFUN>(xv.z, a.up); gs.w += gda_g<GFUN>(xv.w, a.up);
                } else {
                    reinterpret_cast<float4*>(ys)[idx] = yo;
                }
            }
        }
        if (DUAL) {                                          // rows of the warp (lanes with the same quad), then the warps
#pragma unroll
            for (int o = 2; o < 32; o <<= 1) {
                gs.x += __shfl_xor_sync(0xffffffffu, gs.x, o); gs.y += __shfl_xor_sync(0xffffffffu, gs.y, o);
                gs.z += __shfl_xor_sync(0xffffffffu, gs.z, o); gs.w += __shfl_xor_sync(0xffffffffu, gs.w, o);
            }
            if (lane < 2) *reinterpret_cast<float4*>(&s_gred[warp][4 * lane]) = gs;
            __syncthreads();
            if (threadIdx.x < SLAB_S) {
                float t = s_gred[0][threadIdx.x];
                for (int w = 1; w < warps; ++w) t += s_gred[w][threadIdx.x];
                s_mu[threadIdx.x] += a.up.beta * t;          // mu^{t+1} = mu^t + beta_s sum_i g(x_i^t)
            }
        }
        __syncthreads();
        float* tmp = xa; xa = xb; xb = tmp;
        xq = reinterpret_cast<const char*>(xa) + 16 * q;
    }

    // ---- write the state back ----
    for (int e = threadIdx.x; e < a.n * 2; e += blockDim.x) {
        const int row = e >> 1, qq = e & 1;
        if (b0 + 4 * qq < a.B) {
            const size_t off = (size_t)row * a.B + b0 + 4 * qq;
            *reinterpret_cast<float4*>(a.x_out + off) = reinterpret_cast<const float4*>(xa)[e];
            if (!DUAL) *reinterpret_cast<float4*>(a.y + off) = reinterpret_cast<const float4*>(ys)[e];
        }
    }
    if (DUAL && threadIdx.x < SLAB_S && b0 + (int)threadIdx.x < a.B) a.mu_out[b0 + threadIdx.x] = s_mu[threadIdx.x];

    // ---- S5: exact objective of x_hat = [x > 1/2] for the slab's restarts: sum_i x_hat_i ((Q_off x_hat)_i + c'_i) ----
    acc_t obj4[4] = {0, 0, 0, 0};
    for (int i = 0; i < a.groups_per_warp; ++i) {
        const int g = slab_group(i, warp, warps);
        if (g >= a.n_groups) break;
        const int p0 = __ldg(a.goff + g) >> 2, p1 = __ldg(a.goff + g + 1) >> 2;
        const int row = __ldg(a.grow + g * SLAB_ROWS + r);
        float sf[4] = {0.f, 0.f, 0.f, 0.f};                  // fp32 row sums of val2 * x_hat_j (as spmm_score)
        int si[4] = {0, 0, 0, 0};
        for (int ps = p0; ps < p1; ++ps) {
            const SlabPass e = slab_fetch<COMPACT>(a, cst, ps, r);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float4 gv = *reinterpret_cast<const float4*>(xq + e.off[u]);
                if (INTEGRAL) {
                    const int vi = __float2int_rn(e.val[u]);
                    si[0] += gv.x > 0.5f ? vi : 0; si[1] += gv.y > 0.5f ? vi : 0;
                    si[2] += gv.z > 0.5f ? vi : 0; si[3] += gv.w > 0.5f ? vi : 0;
                } else {
                    const float v = e.val[u];
                    sf[0] += gv.x > 0.5f ? v : 0.f; sf[1] += gv.y > 0.5f ? v : 0.f;
                    sf[2] += gv.z > 0.5f ? v : 0.f; sf[3] += gv.w > 0.5f ? v : 0.f;
                }
            }
        }
        if (row >= 0) {
            const float4 xi = reinterpret_cast<const float4*>(xa)[row * 2 + q];
            const float cp = cps[row];
            const bool on[4] = {xi.x > 0.5f, xi.y > 0.5f, xi.z > 0.5f, xi.w > 0.5f};
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (!on[u]) continue;
                if (INTEGRAL) obj4[u] += (long long)(si[u] / 2) + (long long)__float2int_rn(cp);   // val2 = 2 Q_ij: even
                else obj4[u] += 0.5 * (double)sf[u] + (double)cp;
            }
        }
    }
    // rows of the warp: lanes with the same quad, in a fixed butterfly order; then the warps in index order
#pragma unroll
    for (int o = 2; o < 32; o <<= 1)
#pragma unroll
        for (int u = 0; u < 4; ++u) obj4[u] += __shfl_xor_sync(0xffffffffu, obj4[u], o);
    if (lane < 2)
#pragma unroll
        for (int u = 0; u < 4; ++u) red[warp * SLAB_S + 4 * lane + u] = obj4[u];
    __syncthreads();
    double my_best = CUDART_INF_SLAB;
    if (threadIdx.x < SLAB_S) {
        const int b = b0 + threadIdx.x;
        int imp = 0;
        if (b < a.B_eval) {
            acc_t t = red[threadIdx.x];
            for (int w = 1; w < warps; ++w) t += red[w * SLAB_S + threadIdx.x];
            const double v = (double)t;
            double best = a.best_obj[b];
            imp = v < best;
            if (imp) { best = v; a.best_obj[b] = v; }
            a.improved[b] = imp;
            my_best = best;
        }
        s_imp[threadIdx.x] = imp;
    }
    if (warp == 0) {                                         // ticket of the evaluation (see finalize_kernel)
        for (int o = 4; o > 0; o >>= 1) my_best = fmin(my_best, __shfl_xor_sync(0xffffffffu, my_best, o));
        const int any = __any_sync(0xffffffffu, threadIdx.x < SLAB_S && s_imp[threadIdx.x & 7]);
        if (lane == 0) {
            a.block_min[blockIdx.x] = my_best;
            if (any) atomicOr(&a.st->imp_accum, 1u);
            __threadfence();
            s_last = atomicAdd(&a.st->ticket, 1u) == gridDim.x - 1 ? 1u : 0u;
        }
    }
    __syncthreads();
    // ---- commit x_hat of the improved restarts (8 bytes per row, masked) ----
    uint64_t mask = 0;
#pragma unroll
    for (int u = 0; u < SLAB_S; ++u) mask |= s_imp[u] ? (0xFFull << (8 * u)) : 0ull;
    if (mask) {
        for (int row = threadIdx.x; row < a.n; row += blockDim.x) {
            const float4 v0 = reinterpret_cast<const float4*>(xa)[row * 2], v1 = reinterpret_cast<const float4*>(xa)[row * 2 + 1];
            const uint64_t bits = (uint64_t)(v0.x > 0.5f) | ((uint64_t)(v0.y > 0.5f) << 8) | ((uint64_t)(v0.z > 0.5f) << 16) |
                                  ((uint64_t)(v0.w > 0.5f) << 24) | ((uint64_t)(v1.x > 0.5f) << 32) | ((uint64_t)(v1.y > 0.5f) << 40) |
                                  ((uint64_t)(v1.z > 0.5f) << 48) | ((uint64_t)(v1.w > 0.5f) << 56);
            uint8_t* dst = a.x_bin + (size_t)row * a.B + b0;
            if (b0 + SLAB_S <= a.B && (a.B & 7) == 0) {       // aligned 8-byte read-modify-write
                uint64_t* d8 = reinterpret_cast<uint64_t*>(dst);
                *d8 = (*d8 & ~mask) | (bits & mask);
            } else {
                for (int u = 0; u < SLAB_S; ++u)
                    if (b0 + u < a.B && s_imp[u]) dst[u] = (uint8_t)((bits >> (8 * u)) & 1u);
            }
        }
    }
    if (s_last && warp == 0) {                               // every other block has finished (and read st->t long ago)
        __threadfence();
        double m = CUDART_INF_SLAB;
        for (int kk = lane; kk < (int)gridDim.x; kk += 32) m = fmin(m, __ldcg(a.block_min + kk));
        for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (lane == 0) {
            const uint32_t kk = a.st->n_eval;
            if (a.trace_best && (int)kk < a.trace_cap) { a.trace_best[kk] = m; a.trace_ns[kk] = slab_globaltimer_ns(); }
            a.st->n_eval = kk + 1;
            a.st->t = t0 + (uint32_t)a.len;
            a.st->any_improved = atomicExch(&a.st->imp_accum, 0u);
            a.st->ticket = 0;
        }
    }
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

// PDBO-s, start of a run: S^0 = sum_i g(x_i^0) per restart into the fixed-point accumulators, block sums of 8 rows like the
// step kernels' (ScalarDual in gda_internal.cuh)
template <int GFUN>
__global__ void __launch_bounds__(THREADS)
dual_init_kernel(int n, int B, const float* __restrict__ x, UpdParams up, ScalarDual sd) {
    __shared__ float4 gred[WARPS][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int row = blockIdx.x * WARPS + warp;
    const bool active = 4 * (blockIdx.y * 32 + lane) < B;
    const int c4 = active ? blockIdx.y * 32 + lane : B / 4 - 1;
    float4 gs = make_float4(0.f, 0.f, 0.f, 0.f);
    if (row < n && active) {
        const float4 xv = ldg4(x + (size_t)row * B + 4 * c4);
        gs = make_float4(gda_g<GFUN>(xv.x, up), gda_g<GFUN>(xv.y, up), gda_g<GFUN>(xv.z, up), gda_g<GFUN>(xv.w, up));
    }
    scalar_dual_finish<WARPS>(gs, gred, warp, lane, active, c4, blockIdx.x, sd);
}

template <int MODE, bool DUAL>
gda_status launch_step(gda_problem* p, int32_t B, const float* x, float* y, float* xn, const UpdParams& up,
                       const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s, int64_t* launches) {
    const int chunks = (B / 4 + 31) / 32;
    if (MODE == 0 && !DUAL && B <= 64 && !split_all_rows(p, B)) {   // few restarts: several rows per warp
        int G = 1;
        while (4 * G < B) G <<= 1;
        const int split_log2 = narrow_split_log2(p, B);
        const int rows_per_block = NARROW_WARPS * (32 / (G << split_log2));
        const unsigned grid = (unsigned)((p->n + rows_per_block - 1) / rows_per_block);
#define GDA_NW_CASE(GG) case GG: \
        if (up.gfun == GDA_G_QUADRATIC) spmm_step_narrow<GDA_G_QUADRATIC, GG><<<grid, 32 * NARROW_WARPS, 0, s>>>(p->n, B, p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, st, t_off, split_log2); \
        else spmm_step_narrow<GDA_G_ENTROPY, GG><<<grid, 32 * NARROW_WARPS, 0, s>>>(p->n, B, p->d_rowptr, p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, st, t_off, split_log2); break;
        switch (G) { GDA_NW_CASE(1) GDA_NW_CASE(2) GDA_NW_CASE(4) GDA_NW_CASE(8) GDA_NW_CASE(16) default: break; }
#undef GDA_NW_CASE
        if (launches) ++*launches;
        GDA_CUDA_TRY(cudaGetLastError());
        return GDA_OK;
    }
    // A launch of few warps that each walk a long row (small n, high degree, one or two chunks of restarts) is bound by the
    // latency of the serial walk: every row then goes through the row-split kernel with slices of 8 entries instead.
    if (split_all_rows(p, B)) {
        const unsigned grid = (unsigned)(p->n * chunks);
        if (up.gfun == GDA_G_QUADRATIC)
            spmm_step_split<GDA_G_QUADRATIC, MODE, DUAL><<<grid, THREADS, 0, s>>>(p->n, nullptr, B, chunks, p->d_rowptr,
                p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, sd, st, t_off, 8);
        else
            spmm_step_split<GDA_G_ENTROPY, MODE, DUAL><<<grid, THREADS, 0, s>>>(p->n, nullptr, B, chunks, p->d_rowptr,
                p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, sd, st, t_off, 8);
        if (launches) ++*launches;
        GDA_CUDA_TRY(cudaGetLastError());
        return GDA_OK;
    }
    const int n_light = p->d_light_rows ? p->n_light : p->n;
    constexpr int WW = warp_kernel_warps(DUAL), WTHREADS = 32 * WW;
    const int light_blocks = (n_light + WW - 1) / WW;
    const bool pf = MODE == 0 && !DUAL && 12.0 * (double)p->n * (double)B > 0.8 * (double)p->l2_bytes;   // the streaming switch (see spmm_step_warp)
    if (n_light > 0) {
        const dim3 grid((unsigned)light_blocks, (unsigned)chunks);
        const int32_t* row_list = (DUAL && p->d_local_rows && p->opt_row_grouping) ? p->d_local_rows : p->d_light_rows;   // PDBO-s: rows grouped by adjacency
#define GDA_SP_ARGS n_light, row_list, B, p->d_rowptr, p->d_col, p->d_val2, p->d_ell, p->d_cprime, x, y, xn, up, sd, st, t_off
#define GDA_SP_PF(G, E) do { if (pf) spmm_step_warp<G, MODE, E, DUAL, (MODE == 0 && !DUAL)><<<grid, WTHREADS, 0, s>>>(GDA_SP_ARGS); \
                             else spmm_step_warp<G, MODE, E, DUAL, false><<<grid, WTHREADS, 0, s>>>(GDA_SP_ARGS); } while (0)
#define GDA_SP_CASE(E) \
        if (up.gfun == GDA_G_QUADRATIC) GDA_SP_PF(GDA_G_QUADRATIC, E); else GDA_SP_PF(GDA_G_ENTROPY, E)
        if (p->d_ell) { GDA_SP_CASE(true); } else { GDA_SP_CASE(false); }
#undef GDA_SP_PF
#undef GDA_SP_CASE
#undef GDA_SP_ARGS
        if (launches) ++*launches;
    }
    if (p->n_heavy > 0) {
        const unsigned grid = (unsigned)(p->n_heavy * chunks);
        ScalarDual sdh = sd;
        if (n_light > 0) sdh.advance = 0;                     // the launch above closes the multiplier update
        if (up.gfun == GDA_G_QUADRATIC)
            spmm_step_split<GDA_G_QUADRATIC, MODE, DUAL><<<grid, THREADS, 0, s>>>(p->n_heavy, p->d_heavy_rows, B, chunks, p->d_rowptr,
                p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, sdh, st, t_off, 32);
        else
            spmm_step_split<GDA_G_ENTROPY, MODE, DUAL><<<grid, THREADS, 0, s>>>(p->n_heavy, p->d_heavy_rows, B, chunks, p->d_rowptr,
                p->d_col, p->d_val2, p->d_cprime, x, y, xn, up, sdh, st, t_off, 32);
        if (launches) ++*launches;
    }
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

}  // namespace

int sparse_heavy_threshold() { return HEAVY_DEG; }

// shared-memory opt-in of the slab kernels on the handle's device; called at create (never inside a capture)
template <int GFUN, bool INTEGRAL, bool COMPACT>
static gda_status slab_opt_in() {
    GDA_CUDA_TRY(cudaFuncSetAttribute(spmm_chunk_slab<GFUN, INTEGRAL, COMPACT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SLAB_SMEM_LIMIT));
    GDA_CUDA_TRY(cudaFuncSetAttribute(spmm_chunk_slab<GFUN, INTEGRAL, COMPACT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SLAB_SMEM_LIMIT));
    return GDA_OK;
}
gda_status sparse_configure(gda_problem*) {
    GDA_TRY((slab_opt_in<GDA_G_QUADRATIC, true, true>()));   GDA_TRY((slab_opt_in<GDA_G_QUADRATIC, true, false>()));
    GDA_TRY((slab_opt_in<GDA_G_QUADRATIC, false, true>()));  GDA_TRY((slab_opt_in<GDA_G_QUADRATIC, false, false>()));
    GDA_TRY((slab_opt_in<GDA_G_ENTROPY, true, true>()));     GDA_TRY((slab_opt_in<GDA_G_ENTROPY, true, false>()));
    GDA_TRY((slab_opt_in<GDA_G_ENTROPY, false, true>()));    GDA_TRY((slab_opt_in<GDA_G_ENTROPY, false, false>()));
    return GDA_OK;
}

gda_status sparse_step(gda_problem* p, int32_t B, const float* x, float* y, float* xn, const UpdParams& up,
                       const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s, int64_t* launches) {
    if (sd.mu) return launch_step<0, true>(p, B, x, y, xn, up, sd, st, t_off, s, launches);
    return launch_step<0, false>(p, B, x, y, xn, up, sd, st, t_off, s, launches);
}

gda_status sparse_dual_init(gda_problem* p, int32_t B, const float* x, int32_t gfun, float log_eps, unsigned long long* gacc, cudaStream_t s,
                            int64_t* launches) {
    UpdParams up{};
    up.gfun = gfun; up.log_eps = log_eps;                      // the entropy g clamps at log_eps (reading R4)
    ScalarDual sd;
    sd.gacc_next = gacc; sd.B = B;
    const dim3 grid((unsigned)((p->n + WARPS - 1) / WARPS), (unsigned)((B / 4 + 31) / 32));
    if (gfun == GDA_G_QUADRATIC) dual_init_kernel<GDA_G_QUADRATIC><<<grid, THREADS, 0, s>>>(p->n, B, x, up, sd);
    else dual_init_kernel<GDA_G_ENTROPY><<<grid, THREADS, 0, s>>>(p->n, B, x, up, sd);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
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

// ---- slab path, host side ------------------------------------------------------------------------------------------
// Largest n whose slab state (x, x, y: 96 B per row; c': 4 B) and reduction scratch fit the 227 KB a CTA may use
static size_t slab_smem_bytes(int n, int warps, int compact_passes) {       // compact_passes < 0: general structure (global memory)
    const size_t nrow = (size_t)n + (compact_passes >= 0 ? 4 : 0);
    return (2 * nrow * SLAB_S + (size_t)n * SLAB_S + ((n + 3) & ~3)) * sizeof(float) + (size_t)warps * SLAB_S * sizeof(double) +
           (compact_passes >= 0 ? (size_t)compact_passes * SLAB_ROWS * sizeof(uint2) : 0);
}

// Build the sliced-ELL structure described above spmm_chunk_slab.  Called at create with the off-diagonal CSR
// (val2 = 2 Q_ij).  Leaves p->slab_* null when n is too large for the slab kernel.
gda_status sparse_build_slab(gda_problem* p, const std::vector<int32_t>& rowptr, const std::vector<int32_t>& col,
                             const std::vector<float>& val2) {
    const int n = p->n;
    if (slab_smem_bytes(n, 32, -1) > (size_t)SLAB_SMEM_LIMIT) return GDA_OK;
    // rows sorted by degree (descending, stable): the rows that share passes have similar lengths, so little padding
    std::vector<int32_t> order(n);
    for (int i = 0; i < n; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return rowptr[a + 1] - rowptr[a] > rowptr[b + 1] - rowptr[b]; });
    // 0. which rows share a quad.  A quad's schedule is at least as long as its longest row AND as the largest number of
    //    entries its four rows have in one column class (col mod 4: every pass serves each class once), and with random
    //    columns the second bound is the larger one (48-entry rows: about 55).  So inside windows of 128 rows of similar
    //    degree the quads are put together greedily such that the class sums stay level.
    {
        std::vector<std::array<int, 4>> cls(n);
        for (int i = 0; i < n; ++i) {
            cls[i] = {0, 0, 0, 0};
            for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) if (val2[k] != 0.0f) ++cls[i][col[k] & 3];
        }
        constexpr int WINDOW = 128;          // config 2, us per step: no balancing 8.48, windows of 16 / 32 / 64 / 128 / 256 / 800 rows 8.21 / 8.24 / 8.15 / 8.09 / 8.22 / 8.79
        std::vector<int32_t> balanced;
        balanced.reserve(n);
        for (int w0 = 0; w0 < n; w0 += WINDOW) {
            std::vector<int32_t> pool(order.begin() + w0, order.begin() + std::min(n, w0 + WINDOW));
            while (!pool.empty()) {
                std::array<int, 4> sum = cls[pool[0]];
                balanced.push_back(pool[0]);
                pool.erase(pool.begin());
                for (int j = 1; j < 4 && !pool.empty(); ++j) {
                    size_t best = 0; long best_score = -1;
                    for (size_t q = 0; q < pool.size(); ++q) {
                        long mx = 0, sq = 0;
                        for (int c = 0; c < 4; ++c) { const long v = sum[c] + cls[pool[q]][c]; mx = std::max(mx, v); sq += v * v; }
                        const long score = mx * 1000000L + sq;
                        if (best_score < 0 || score < best_score) { best_score = score; best = q; }
                    }
                    for (int c = 0; c < 4; ++c) sum[c] += cls[pool[best]][c];
                    balanced.push_back(pool[best]);
                    pool.erase(pool.begin() + best);
                }
            }
        }
        order.swap(balanced);
    }
    // 1. quads of four rows of similar degree.  The four rows of a quad share every LDS.128 pass: order their entries
    //    such that the four columns of a pass differ mod 4 (one 32-byte row of x per bank group).  Greedy: per pass, the
    //    assignment of distinct classes to the rows that uses up the most entries, ties to the largest remaining
    //    queues; zero-valued padding elsewhere.
    struct Quad { int32_t row[4]; std::vector<int2> sched[4]; size_t len = 0; };
    const int n_quads = (n + 3) / 4;
    std::vector<Quad> quads(n_quads);
    int64_t real_entries = 0;
    static const int perms[24][4] = {{0,1,2,3},{0,1,3,2},{0,2,1,3},{0,2,3,1},{0,3,1,2},{0,3,2,1},{1,0,2,3},{1,0,3,2},
        {1,2,0,3},{1,2,3,0},{1,3,0,2},{1,3,2,0},{2,0,1,3},{2,0,3,1},{2,1,0,3},{2,1,3,0},{2,3,0,1},{2,3,1,0},
        {3,0,1,2},{3,0,2,1},{3,1,0,2},{3,1,2,0},{3,2,0,1},{3,2,1,0}};
    for (int qd = 0; qd < n_quads; ++qd) {
        Quad& Q4 = quads[qd];
        std::vector<int2> queue[4][4];                          // [row of the quad][column class]
        int remaining = 0;
        for (int j = 0; j < 4; ++j) {
            const int row = 4 * qd + j < n ? order[4 * qd + j] : -1;
            Q4.row[j] = row;
            if (row < 0) continue;
            for (int k = rowptr[row]; k < rowptr[row + 1]; ++k) {
                if (val2[k] == 0.0f) continue;                  // explicit zeros contribute nothing
                int2 e;
                e.x = col[k] * (SLAB_S * 4);
                std::memcpy(&e.y, &val2[k], 4);
                queue[j][col[k] & 3].push_back(e);
                ++remaining;
            }
        }
        real_entries += remaining;
        while (remaining > 0) {
            int best = 0; long best_score = -1;
            for (int pi = 0; pi < 24; ++pi) {
                long used = 0, left = 0;
                for (int j = 0; j < 4; ++j) { const size_t sz = queue[j][perms[pi][j]].size(); used += sz > 0; left += (long)sz; }
                const long score = used * 1000000L + left;
                if (score > best_score) { best_score = score; best = pi; }
            }
            for (int j = 0; j < 4; ++j) {
                const int c = perms[best][j];
                int2 e;
                if (!queue[j][c].empty()) { e = queue[j][c].back(); queue[j][c].pop_back(); --remaining; }
                else { e.x = -1 - c; e.y = 0; }                                    // padding of class c, value 0 (resolved below)
                Q4.sched[j].push_back(e);
            }
            ++Q4.len;
        }
    }
    // 2. quads sorted by the length of their schedule, four of them per 16-row group (a warp walks them in lockstep,
    //    so a group costs its longest quad)
    std::vector<int32_t> qorder(n_quads);
    for (int i = 0; i < n_quads; ++i) qorder[i] = i;
    std::stable_sort(qorder.begin(), qorder.end(), [&](int a, int b) { return quads[a].len > quads[b].len; });
    const int n_groups = (n_quads + 3) / 4;
    std::vector<int32_t> goff(n_groups + 1, 0), grow((size_t)n_groups * SLAB_ROWS, -1);
    std::vector<int2> ent;
    for (int g = 0; g < n_groups; ++g) {
        size_t len = 0;
        for (int h = 0; h < 4; ++h)
            if (4 * g + h < n_quads) len = std::max(len, quads[qorder[4 * g + h]].len);
        len = (len + 3) & ~(size_t)3;                           // the kernel walks 4 slots at a time
        for (int h = 0; h < 4; ++h)
            for (int j = 0; j < 4; ++j)
                if (4 * g + h < n_quads) grow[(size_t)g * SLAB_ROWS + 4 * h + j] = quads[qorder[4 * g + h]].row[j];
        for (size_t k = 0; k < len; ++k)
            for (int r = 0; r < SLAB_ROWS; ++r) {
                int2 e;
                const int h = r >> 2, j = r & 3;
                if (4 * g + h < n_quads && k < quads[qorder[4 * g + h]].sched[j].size()) e = quads[qorder[4 * g + h]].sched[j][k];
                else { e.x = -1 - (int)((k + r) & 3); e.y = 0; }
                ent.push_back(e);
            }
        goff[g + 1] = goff[g] + (int32_t)len;
    }
    // one more pass of padding that belongs to no group: what the "next pass" prefetch of the last pass reads
    for (int k = 0; k < 4 * SLAB_ROWS; ++k) { int2 e; e.x = -1 - (k & 3); e.y = 0; ent.push_back(e); }
    p->slab_groups = n_groups;
    p->slab_slots = goff[n_groups] + 4;
    p->slab_real = real_entries;
    // compact form: every non-zero |val2| is the same number, columns (and the four zero rows n .. n+3 that padding
    // entries gather) fit 12 bits, and the structure fits shared memory next to the state
    uint32_t cbits = 0;
    bool compact = n + 4 <= 4096;
    for (size_t k = 0; k < ent.size() && compact; ++k) {
        if (ent[k].x < 0) continue;
        const uint32_t mag = (uint32_t)ent[k].y & 0x7FFFFFFFu;
        if (cbits == 0) cbits = mag;
        compact = mag == cbits;
    }
    const int n_pass = p->slab_slots / 4;
    compact = compact && cbits != 0 && slab_smem_bytes(n, 32, n_pass) <= (size_t)SLAB_SMEM_LIMIT;
    if (compact) {
        std::vector<uint16_t> e16((size_t)n_pass * SLAB_ROWS * 4);
        for (int ps = 0; ps < n_pass; ++ps)
            for (int r = 0; r < SLAB_ROWS; ++r)
                for (int u = 0; u < 4; ++u) {
                    const int2 e = ent[((size_t)ps * 4 + u) * SLAB_ROWS + r];
                    // padding of class c gathers the zero row n + j with (n + j) mod 4 == c
                    const uint32_t colv = e.x < 0 ? (uint32_t)(n + ((((-1 - e.x) - n) % 4) + 4) % 4) : (uint32_t)(e.x / (SLAB_S * 4));
                    e16[((size_t)ps * SLAB_ROWS + r) * 4 + u] = (uint16_t)(colv | (((uint32_t)e.y >> 31) << 15));
                }
        GDA_CUDA_TRY(cudaMalloc((void**)&p->d_slab_ent16, e16.size() * sizeof(uint16_t)));
        GDA_CUDA_TRY(cudaMemcpy(p->d_slab_ent16, e16.data(), e16.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
        p->slab_cbits = cbits;
        p->slab_passes = n_pass;
    }
    // general form: padding gathers a real row of the wanted class (value 0)
    for (auto& e : ent) if (e.x < 0) e.x = std::min(-1 - e.x, n - 1) * (SLAB_S * 4);
    const size_t bytes = std::max<size_t>(ent.size(), 1) * sizeof(int2);
    GDA_CUDA_TRY(cudaMalloc((void**)&p->d_slab_ent, bytes));
    if (!ent.empty()) GDA_CUDA_TRY(cudaMemcpy(p->d_slab_ent, ent.data(), ent.size() * sizeof(int2), cudaMemcpyHostToDevice));
    GDA_CUDA_TRY(cudaMalloc((void**)&p->d_slab_goff, goff.size() * sizeof(int32_t)));
    GDA_CUDA_TRY(cudaMemcpy(p->d_slab_goff, goff.data(), goff.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    GDA_CUDA_TRY(cudaMalloc((void**)&p->d_slab_grow, grow.size() * sizeof(int32_t)));
    GDA_CUDA_TRY(cudaMemcpy(p->d_slab_grow, grow.data(), grow.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    return GDA_OK;
}

// Is the slab kernel the faster way to run a chunk at this B?  Its step costs the shared-memory gathers of one CTA
// (slots x 16 rows x 32 B at 128 B per clock) times the number of waves of B / 8 CTAs; the streaming kernel one launch
// (about 2.5 us) or its L2 gathers (nnz x B x 4 B at about 13 TB/s, measured on config 2), whichever is larger.
static bool slab_wanted(const gda_problem* p, int32_t B) {
    if (!p->d_slab_ent || p->slab_mode < 0) return false;
    if (p->slab_mode > 0) return true;
    const double ctas = (B + SLAB_S - 1) / SLAB_S, waves = std::ceil(ctas / p->num_sms);
    const double t_slab = waves * (1.3 * (double)p->slab_slots * SLAB_ROWS * 32.0 / 128.0 / 1.9e3 + 0.3);   // us (1.3: structure, own state, barriers; config 2: 8.4)
    // streaming step, us: the gathers out of the L2 at 13 TB/s, a launch, and -- few warps that each walk a long row -- the
    // latency of that walk (measured on config 2's graph, see split_all_rows)
    const double gather_us = (double)p->nnz * B * 4.0 / 13e6;
    const double deg = (double)p->nnz / std::max(p->n, 1) / (B <= 64 && !split_all_rows(p, B) ? (double)(1 << narrow_split_log2(p, B)) : 1.0);   // entries one lane group walks
    const double t_stream = split_all_rows(p, B) ? 3.2 + 1.1 * gather_us : std::max(std::max(2.5, gather_us), 1.5 + 0.15 * deg);
    return t_slab < t_stream;
}

// One launch = `len` steps + the evaluation, when the slab kernel applies; *done = 0 when it does not.
gda_status sparse_chunk_slab(gda_problem* p, int32_t B_eval, int32_t B, int32_t len, const float* x_in, float* x_out, float* y,
                             const float* mu_in, float* mu_out, const UpdParams& up, cudaStream_t s, int64_t* launches, int* done) {
    *done = 0;
    if (!slab_wanted(p, B)) return GDA_OK;
    Workspace& ws = p->ws;
    const int per_warp = (p->slab_groups + 31) / 32;
    const int warps = std::max(1, (p->slab_groups + per_warp - 1) / per_warp);
    const bool compact = p->d_slab_ent16 != nullptr;
    SlabArgs a{};
    a.n = p->n; a.B = B; a.B_eval = B_eval; a.len = len; a.n_groups = p->slab_groups; a.groups_per_warp = per_warp; a.n_pass = p->slab_slots / 4;
    a.ent = p->d_slab_ent; a.ent16 = reinterpret_cast<const uint2*>(p->d_slab_ent16); a.cbits = p->slab_cbits;
    a.goff = p->d_slab_goff; a.grow = p->d_slab_grow; a.cprime = p->d_cprime;
    a.x_in = x_in; a.x_out = x_out; a.y = y; a.mu_in = mu_in; a.mu_out = mu_out; a.up = up; a.st = ws.state;
    a.best_obj = ws.best_obj; a.improved = ws.improved; a.x_bin = ws.x_bin; a.block_min = ws.block_min;
    a.trace_best = ws.trace_best; a.trace_ns = ws.trace_ns; a.trace_cap = ws.trace_cap;
    const unsigned grid = (unsigned)((B + SLAB_S - 1) / SLAB_S);
    const size_t smem = slab_smem_bytes(p->n, warps, compact ? a.n_pass : -1);
    const bool quad = up.gfun == GDA_G_QUADRATIC;
#define GDA_SLAB_LAUNCH(G, I, C) do { if (mu_in) spmm_chunk_slab<G, I, C, true><<<grid, warps * 32, smem, s>>>(a); \
                                      else spmm_chunk_slab<G, I, C, false><<<grid, warps * 32, smem, s>>>(a); } while (0)
#define GDA_SLAB_IC(G) do { if (p->integral) { if (compact) GDA_SLAB_LAUNCH(G, true, true); else GDA_SLAB_LAUNCH(G, true, false); } \
                            else { if (compact) GDA_SLAB_LAUNCH(G, false, true); else GDA_SLAB_LAUNCH(G, false, false); } } while (0)
    if (quad) GDA_SLAB_IC(GDA_G_QUADRATIC); else GDA_SLAB_IC(GDA_G_ENTROPY);
#undef GDA_SLAB_IC
#undef GDA_SLAB_LAUNCH
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    *done = 1;
    return GDA_OK;
}
