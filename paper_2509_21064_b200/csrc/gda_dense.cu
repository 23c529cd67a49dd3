// gda_dense.cu -- S2 + S4 for dense QUBO: tcgen05 / TMA / TMEM GEMM gradient with the GDA update fused
// into the epilogue.
//
//   G = 2 Q_off X + c' 1^T          (reading R1)
// computed with the CENTRED bf16 operand z = x - 1/2 (reading R13):  G = 2 Q_off z + (Q_off 1 + c').
//
// GEMM shape (both operands K-major, the layout tcgen05 takes without transposition):
//   D[b][i] = sum_k Zt[b][k] * Qoff[i][k]        M = restarts b, N = variables i, K = variables k
//   A = Zt   bf16 [B][n]  (the transposed, centred copy of X; double-buffered: step t reads zt_in while
//                          its epilogue writes zt_out for step t+1 -- Jacobi update, Eq. 6)
//   B = Qoff bf16 [n][n]  (symmetric, zero diagonal)
//   D fp32 in TMEM: lane = restart b (128 per tile), column = variable i (256 per tile), two accumulator
//   stages (2 x 256 = 512 columns) so the epilogue of tile t overlaps the MMAs of tile t+1.
// With lanes = restarts the epilogue's accesses to the fp32 state X, Y ([n][B]) are coalesced 128-byte
// rows per warp; the next bf16 operand ([B][n], a restart's variables contiguous) leaves through a swizzled staging
// tile per warp in shared memory and TMA stores of 32 x 64 boxes (whole 128-byte lines).
//
// Warp roles (384 threads, one persistent CTA per SM): warp 0 TMA producer, warp 1 MMA issuer (one
// elected thread), warp 2 TMEM allocator, warps 4-11 epilogue (two warpgroups, half of the tile's columns each).
//
// Operand feed (measured, profiles/): with one CTA per 128 x 256 tile the kernel was bound by operand delivery, not
// by the tensor pipe -- 48 KB per CTA and 512-cycle k-block out of L2, about 1.6 GB per step, which is what the L2
// can deliver in the time the step took.  Hence, when the shape allows:
//  * CTA PAIRS (tcgen05 cta_group::2, M = 256): each CTA stages its own 128 rows of A and HALF of the Q tile, the
//    tensor cores of both SMs read both halves; 32 KB per CTA and k-block, 6 stages in flight.  The leader (even rank)
//    issues the MMAs; both CTAs' TMA loads signal the leader's full barrier; tcgen05.commit multicasts "slot free" and
//    "accumulator ready"; the peer's epilogue warps release the accumulator on the leader's barrier through the
//    cluster address space.  Each CTA keeps its 128 rows of the accumulator in its own TMEM: same epilogue.
//  * TWO PAIRS PER CLUSTER (PM = 1, PN = 2, cluster of 4) that work on the same 256 restarts and adjacent blocks of 256
//    variables: each CTA loads half of its A rows and TMA-multicasts them to its counterpart in the other pair
//    (24 KB per CTA and k-block).  A slot is reused when BOTH pairs have retired it (empty barrier count 2, every
//    leader's commit goes to all four CTAs).
//  * FOUR PAIRS PER CLUSTER (PM = PN = 2, cluster of 8): pairs (pm, pn) on restart block pm and variable block pn.  The
//    A rows of a CTA are shared along pn and its half of the Q tile along pm; every CTA loads one 64-row box of each
//    and multicasts it to its partner (16 KB of L2 reads per CTA and k-block).  The step is bound by what the L2 can
//    deliver while 128 SMs stream operands, so every byte not read twice shortens it.
// B an odd multiple of 128 runs single CTAs (CG = 1); n not a multiple of 512 runs pairs without the multicast; B not a
// multiple of 512 runs clusters of two pairs.
//
// Tile schedule: work units of (PM x CG x 128 restarts) x (PN x 256 variables) are dealt round-robin to the clusters.
// A 128-variable "half" unit does NOT help the tail: measured, an N = 128 MMA takes as long as an N = 256 one (the
// A-operand path of M = 128 rows per SM sets the instruction time), so units always span 256 variables per pair.
#include "gda_internal.cuh"

#include <cuda.h>
#include <cmath>
#include <cstdlib>
#include <vector>

#ifndef GDA_DENSE_STAGES
#define GDA_DENSE_STAGES 6      // pipeline stages of the pair variants (32 KB each)
#endif

namespace {

constexpr int BM = 128, BN = 256, BK = 64, UMMA_K = 16, BBOX = 64;   // BBOX: rows per TMA box (both operands)
constexpr int A_BYTES = BM * BK * 2;
constexpr int NUM_THREADS = 384, EPI_WARP0 = 4, EPI_WARPS = 8;
constexpr int TMEM_COLS = 512;
// epilogue staging of the NEXT bf16 operand: per epilogue warp 32 restarts x 64 variables (128-byte rows, 128-byte swizzle),
// written back by TMA stores as whole 128-byte lines (16-byte stores straight from registers leave half-filled sectors)
constexpr int ZST_COLS = 64, ZST_WARP_BYTES = 32 * ZST_COLS * 2, ZST_BYTES = 8 * ZST_WARP_BYTES;
// per CTA and pipeline stage: its 128 rows of A and its 256 / CG rows of Q; 4 stages of 48 KB or 6 stages of 32 KB
template <int CG> struct Pipe {
    static constexpr int STAGE_BYTES = A_BYTES + (BN / CG) * BK * 2;
    static constexpr int STAGES = CG == 1 ? 4 : GDA_DENSE_STAGES;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + ZST_BYTES + 256 + 1024;   // tiles + operand staging + barriers + alignment slack
};

enum { MODE_STEP = 0, MODE_GRAD = 1, MODE_SCORE = 2, MODE_STEP_S = 3 };   // MODE_STEP_S: PDBO-s step (one multiplier per restart)

// ---- PTX wrappers -------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// try_wait suspends in hardware for a bounded time per call; a wait that never completes is a pipeline bug,
// so trap instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    for (uint32_t spins = 0; !mbar_try_wait(bar, parity); ++spins)
        if (spins > (1u << 26)) __trap();
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
// pair mode: the load lands in THIS CTA's shared memory and signals `bar` given as a shared::cluster address
// (the leader's full barrier), which cta_group::2 allows
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap* map, uint32_t bar_cluster, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar_cluster), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tc_commit_pair(uint32_t bar, uint16_t mask) {      // arrives on `bar` of every CTA in mask
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(bar), "h"(mask) : "memory");
}
// pair mode + multicast: the box lands at the same offset in every CTA of mask and signals, in each of them, the
// barrier at bar's offset in that CTA's pair leader
__device__ __forceinline__ void tma_load_2d_pair_mc(uint32_t dst, const CUtensorMap* map, uint32_t bar_cluster, int c0, int c1, uint16_t mask) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%3, %4}], [%2], %5;"
        ::"r"(dst), "l"(map), "r"(bar_cluster), "r"(c0), "r"(c1), "h"(mask) : "memory");
}
__device__ __forceinline__ void tc_mma_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ uint32_t map_to_cta(uint32_t smem_addr, uint32_t rank) {  // shared::cta -> shared::cluster of `rank`
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t bar_cluster) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar_cluster) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem], bf16 x bf16 -> fp32, issued by one thread
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// 32 lanes x 32 columns of fp32 accumulator -> 32 registers per thread (thread = lane, register = column)
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tc_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
}
// TMA store of one box from shared memory (bulk async-group completion)
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, uint32_t src, int c0, int c1) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
                 ::"l"(map), "r"(src), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major, 128-byte-swizzled shared-memory operand descriptor (rows of 64 bf16 = 128 B, 8-row groups 1024 B apart)
__device__ __forceinline__ uint64_t make_sdesc(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFF) >> 4);          // [0,14)  start address / 16
    d |= (uint64_t)1 << 16;                               // [16,30) leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(1024 >> 4) << 32;                     // [32,46) stride byte offset: 8 rows x 128 B
    d |= (uint64_t)1 << 46;                               // [46,48) descriptor version (sm_100)
    d |= (uint64_t)2 << 61;                               // [61,64) layout: SWIZZLE_128B
    return d;
}
// instruction descriptor, kind::f16: D fp32, A/B bf16, both K-major, N and M of the UMMA
__host__ __device__ constexpr uint32_t make_idesc(int M, int N) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// ---- the fused GEMM + update kernel ----------------------------------------------------------------------
struct DenseArgs {
    int n, B;
    float* x;                    // [n][B] fp32 state, updated in place (each element is owned by one thread)
    float* y;                    // [n][B]
    __nv_bfloat16* zt_out;       // [B][n] centred bf16 operand of the NEXT step
    const float* hvec;           // [n]  Q_off 1 + c'  (constant part of the gradient with the centred operand)
    const float* cprime;         // [n]  c + diag(Q)
    float* gout;                 // MODE_GRAD: [n][B] gradient
    double* partial;             // MODE_SCORE: [n/128][B] partial objective sums
    const float* mu;             // MODE_STEP_S: [B] this step's multipliers
    float* gpart;                // MODE_STEP_S: [n/128][B] sums of g(x_i^t) over each 128-variable share
    UpdParams up;
    const RunState* st;
    uint32_t t_off;
};

// Work unit u of the schedule described at the top: restarts [m0, m0 + 128) of THIS CTA, variables [n0, n0 + 256)
// of its pair.  rank = rank in the cluster = ((pm * PN) + pn) * CG + r.
struct Unit { int m0, n0; };
__device__ __forceinline__ Unit get_unit(int u, int B, int cg, int pm_n, int pn_n, int rank) {
    const int num_msup = B / (BM * cg * pm_n);
    const int pair = rank / cg, r = rank % cg;
    Unit t;
    t.m0 = (((u % num_msup) * pm_n + pair / pn_n) * cg + r) * BM;
    t.n0 = ((u / num_msup) * pn_n + pair % pn_n) * BN;
    return t;
}
__device__ __forceinline__ int num_units(int n, int B, int cg, int pm_n, int pn_n) { return (B / (BM * cg * pm_n)) * (n / (BN * pn_n)); }

template <int MODE, int GFUN, int CG, int PM, int PN>
__global__ void __launch_bounds__(NUM_THREADS, 1)
dense_gemm_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b,
                  const __grid_constant__ CUtensorMap tmap_zo, const DenseArgs args) {
    constexpr int STAGES = Pipe<CG>::STAGES, STAGE_BYTES = Pipe<CG>::STAGE_BYTES;
    constexpr bool STEP = MODE == MODE_STEP || MODE == MODE_STEP_S, SDUAL = MODE == MODE_STEP_S;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;            // SWIZZLE_128B needs 1024 B alignment
    const uint32_t zst_base = smem_base + STAGES * STAGE_BYTES;                  // 1024-byte aligned (stages are multiples of 1 KB)
    const uint32_t bar_base = zst_base + ZST_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + 2 + s); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
    volatile uint32_t* tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int NP = PM * PN;                                                  // pairs per cluster
    constexpr int CSIZE = CG * NP;                                               // CTAs per cluster
    const int rank = CSIZE > 1 ? (int)cluster_ctarank() : 0;
    const int lead = rank & ~(CG - 1);                                           // rank of this CTA's pair leader
    const bool leader = rank == lead;
    const int cluster_id = blockIdx.x / CSIZE, num_clusters = gridDim.x / CSIZE;
    const int units = num_units(args.n, args.B, CG, PM, PN);
    const int num_kb = args.n / BK;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_a) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_b) : "memory");
        if (STEP) asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap_zo) : "memory");
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), NP); }
        for (int s = 0; s < 2; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), CG * EPI_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {                                       // pair mode: the same warp of both CTAs allocates together
        if (CG == 1) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(TMEM_COLS) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "r"(TMEM_COLS) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        }
    }
    tc_fence_before();
    if (CSIZE > 1) cluster_sync_all(); else __syncthreads();      // the peers' barriers exist before anything signals them
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===== TMA producer (both CTAs of a pair: own rows of A, own half of the Q tile) =====
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            constexpr int SLICE = BN / CG;                                        // rows of Q this CTA stages
            constexpr uint32_t BYTES = (uint32_t)(CG * (A_BYTES + SLICE * BK * 2)); // a pair's loads land on its leader's barrier
            for (int u = cluster_id; u < units; u += num_clusters) {
                const Unit t = get_unit(u, args.B, CG, PM, PN, rank);
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);                      // every MMA that read this slot has retired
                    const uint32_t a_dst = smem_base + stage * STAGE_BYTES;
                    if (CG == 1) {
                        mbar_expect_tx(full_bar(stage), BYTES);
                        for (int r = 0; r < BM; r += BBOX)
                            tma_load_2d(a_dst + (uint32_t)r * 128u, &tmap_a, full_bar(stage), kb * BK, t.m0 + r);
                        for (int r = 0; r < SLICE; r += BBOX)
                            tma_load_2d(a_dst + A_BYTES + (uint32_t)r * 128u, &tmap_b, full_bar(stage), kb * BK, t.n0 + r);
                    } else {
                        if (leader) mbar_expect_tx(full_bar(stage), BYTES);
                        const uint32_t lead_bar = map_to_cta(full_bar(stage), (uint32_t)lead);
                        const int pm = (rank / CG) / PN, pn = (rank / CG) % PN, r2 = rank % CG;
                        if (PN == 1) {
                            for (int r = 0; r < BM; r += BBOX)
                                tma_load_2d_pair(a_dst + (uint32_t)r * 128u, &tmap_a, lead_bar, kb * BK, t.m0 + r);
                        } else {                                                  // my share of the A rows, to the pairs along pn
                            static_assert(PN == 1 || BM / PN == BBOX, "one box per share of the A rows");
                            const int share = pn * (BM / PN);
                            uint16_t mask = 0;
#pragma unroll
                            for (int q = 0; q < PN; ++q) mask |= (uint16_t)(1u << ((pm * PN + q) * CG + r2));
                            tma_load_2d_pair_mc(a_dst + (uint32_t)share * 128u, &tmap_a, lead_bar, kb * BK, t.m0 + share, mask);
                        }
                        if (PM == 1) {
                            for (int r = 0; r < SLICE; r += BBOX)
                                tma_load_2d_pair(a_dst + A_BYTES + (uint32_t)r * 128u, &tmap_b, lead_bar, kb * BK,
                                                 t.n0 + r2 * SLICE + r);
                        } else {                                                  // my share of this CTA's half of the Q tile, to the pairs along pm
                            static_assert(PM == 1 || SLICE / PM == BBOX, "one box per share of the Q rows");
                            const int share = pm * (SLICE / PM);
                            uint16_t mask = 0;
#pragma unroll
                            for (int q = 0; q < PM; ++q) mask |= (uint16_t)(1u << ((q * PN + pn) * CG + r2));
                            tma_load_2d_pair_mc(a_dst + A_BYTES + (uint32_t)share * 128u, &tmap_b, lead_bar, kb * BK,
                                                t.n0 + r2 * SLICE + share, mask);
                        }
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
            if (CG > 1)                                                            // every release aimed at this CTA has landed
                for (int i = 0; i < STAGES; ++i) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one thread; pair mode: the leader CTA only) =====
        if (lane == 0 && leader) {
            int stage = 0; uint32_t phase = 0; int it = 0;
            constexpr uint32_t idesc = make_idesc(BM * CG, BN);
            constexpr uint16_t ALL = (uint16_t)((1u << CSIZE) - 1u);
            const uint16_t mine = (uint16_t)(((1u << CG) - 1u) << lead);
            for (int u = cluster_id; u < units; u += num_clusters, ++it) {
#ifdef GDA_DENSE_SERIAL
                const int as = 0;
                const uint32_t aphase = (uint32_t)it & 1u;
#else
                const int as = it & 1;
                const uint32_t aphase = (uint32_t)(it >> 1) & 1u;
#endif
                mbar_wait(tempty_bar(as), aphase ^ 1u);                           // every epilogue warp has drained this accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(as * BN);
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(full_bar(stage), phase);                            // TMA bytes have landed (in both CTAs)
                    tc_fence_after();
                    const uint32_t a_addr = smem_base + stage * STAGE_BYTES;
                    const uint64_t adesc = make_sdesc(a_addr), bdesc = make_sdesc(a_addr + A_BYTES);
#pragma unroll
                    for (int k = 0; k < BK / UMMA_K; ++k) {                        // +32 B per K=16 slice inside the swizzle atom
                        if (CG == 1) tc_mma(d_tmem, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (uint32_t)((kb | k) != 0));
                        else tc_mma_pair(d_tmem, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (uint32_t)((kb | k) != 0));
                    }
                    if (CG == 1) tc_commit(empty_bar(stage)); else tc_commit_pair(empty_bar(stage), ALL);   // slot free, to every CTA of the cluster
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
                if (CG == 1) tc_commit(tfull_bar(as)); else tc_commit_pair(tfull_bar(as), mine);       // accumulator complete (own pair)
            }
        }
    } else if (warp >= EPI_WARP0) {
        // ===== epilogue: TMEM -> registers -> fused GDA update -> global =====
        const int ew = warp - EPI_WARP0;
        const int lane_grp = warp & 3;                      // TMEM lanes 32*lane_grp .. +31 are accessible to this warp
        const int half = ew >> 2;                           // which half of the tile's columns
        const uint32_t tstep = (args.st ? args.st->t : 0u) + args.t_off;
        int it = 0;
        for (int u = cluster_id; u < units; u += num_clusters, ++it) {
            const Unit t = get_unit(u, args.B, CG, PM, PN, rank);
#ifdef GDA_DENSE_SERIAL
            const int as = 0;
            const uint32_t aphase = (uint32_t)it & 1u;
#else
            const int as = it & 1;
            const uint32_t aphase = (uint32_t)(it >> 1) & 1u;
#endif
            const int b = t.m0 + lane_grp * 32 + lane;                            // restart owned by this thread
            constexpr int hcols = BN / 2;                                         // 128 columns per warpgroup
            mbar_wait(tfull_bar(as), aphase);
            tc_fence_after();
            double score = 0.0;
            if (STEP) {
                // Rounds of 16 variables: 32 loads, 16 updates in registers, 32 stores + 32 bytes of the next operand into the
                // staging tile (double buffering with and without setmaxnreg, more warps and bulk-async staging of x, y were
                // all measured: no faster).  PDBO-s (SDUAL): the multiplier is
                // one number per restart, y is neither read nor written, and the thread's sum of g(x_i^t) over its 128
                // variables goes to gpart.
                const int c_first = half * hcols;                                 // this warpgroup's first column in the tile
                float* __restrict__ xp = args.x + (size_t)(t.n0 + c_first) * args.B + b;
                float* __restrict__ yp = args.y + (size_t)(t.n0 + c_first) * args.B + b;
                const uint32_t zst_warp = zst_base + (uint32_t)ew * ZST_WARP_BYTES;  // this warp's staging tile: row = lane
                const uint32_t zst_row = zst_warp + (uint32_t)lane * 128u;
                const uint32_t trow = tmem_base + ((uint32_t)(lane_grp * 32) << 16) + (uint32_t)(as * BN + c_first);
                const int rounds = hcols / 16;
                const float mu_b = SDUAL ? __ldg(args.mu + b) : 0.0f;
                float gsum = 0.0f;
                float xa[16], ya[16];
                auto load16 = [&](float (&xv)[16], float (&yv)[16], int r) {
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        xv[j] = xp[(size_t)(16 * r + j) * args.B];
                        yv[j] = SDUAL ? mu_b : yp[(size_t)(16 * r + j) * args.B];
                    }
                };
                auto round16 = [&](float (&xv)[16], float (&yv)[16], int r) {
                    uint32_t acc[16];
                    tc_ld16(trow + (uint32_t)(16 * r), acc);
                    // constant part of the gradient: lane j (mod 16) fetches column j of the round, broadcast by shuffle
                    // (a per-element load would sit between the stores and serialise: x, y and hvec may alias)
                    const float hv = __ldg(args.hvec + t.n0 + c_first + 16 * r + (lane & 15));
                    tc_wait_ld();
                    // Eq. 6 for 16 elements as independent, branch-free chains; the (rare) perturbation of reading R3 is
                    // applied afterwards behind ONE test -- a branch per element serialises the loop
                    float xt[16];
                    uint32_t band = 0u;
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const float G = fmaf(2.0f, __uint_as_float(acc[j]), __shfl_sync(0xffffffffu, hv, j));
                        if (SDUAL) gsum += gda_g<GFUN>(xv[j], args.up);
                        gda_update_nopert<GFUN>(xv[j], yv[j], G, args.up, xt[j], yv[j]);
                        band |= gda_in_band(xv[j], xt[j], args.up.delta) ? (1u << j) : 0u;
                    }
                    if (band) {
#pragma unroll
                        for (int j = 0; j < 16; ++j)
                            if (band & (1u << j))
                                xt[j] = gda_perturb(xv[j], xt[j], args.up.delta, args.up.seed_mix, tstep,
                                                    (uint32_t)(t.n0 + c_first + 16 * r + j), (uint32_t)b);
                    }
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        xp[(size_t)(16 * r + j) * args.B] = xt[j];
                        if (!SDUAL) yp[(size_t)(16 * r + j) * args.B] = yv[j];
                    }
                    // next operand: 16 bf16 of this restart's row into the warp's staging tile (16-byte chunk c of row l
                    // sits at chunk c ^ (l & 7): the 128-byte swizzle of the store map, and conflict-free); every fourth
                    // round one lane hands the 32 x 64 tile to the TMA unit
                    if ((r & 3) == 0) {
                        if (lane == 0) bulk_wait_read0();                         // the previous tile has left shared memory
                        __syncwarp();
                    }
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        uint32_t pk[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const __nv_bfloat162 z2 = __floats2bfloat162_rn(xt[8 * q + 2 * e] - 0.5f, xt[8 * q + 2 * e + 1] - 0.5f);
                            pk[e] = *reinterpret_cast<const uint32_t*>(&z2);
                        }
                        const uint32_t chunk = (uint32_t)(2 * (r & 3) + q);
                        st_shared_v4(zst_row + ((chunk ^ (uint32_t)(lane & 7)) << 4), pk[0], pk[1], pk[2], pk[3]);
                    }
                    if ((r & 3) == 3) {
                        fence_async_smem();
                        __syncwarp();
                        if (lane == 0) {
                            tma_store_2d(&tmap_zo, zst_warp, t.n0 + c_first + ZST_COLS * (r >> 2), t.m0 + lane_grp * 32);
                            bulk_commit();
                        }
                    }
                };
#pragma unroll 1
                for (int r = 0; r < rounds; ++r) {
                    load16(xa, ya, r);
                    round16(xa, ya, r);
                }
                if (SDUAL) args.gpart[(size_t)((t.n0 + c_first) / 128) * args.B + b] = gsum;
            }
            for (int cb = 0; !STEP && cb < hcols / 32; ++cb) {
                const int col0 = half * hcols + cb * 32;
                const int i0 = t.n0 + col0;
                uint32_t acc[32];
                tc_ld32(tmem_base + ((uint32_t)(lane_grp * 32) << 16) + (uint32_t)(as * BN + col0), acc);
                // the constant part of the gradient for these 32 columns: one coalesced load, lane j holds column j
                // (a per-element load would sit between the stores below and serialise the loop: the compiler must
                // assume that x, y and hvec alias)
                const float hv = __ldg(args.hvec + i0 + lane);
                if (MODE == MODE_GRAD) {
                    tc_wait_ld();
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        args.gout[(size_t)(i0 + j) * args.B + b] = fmaf(2.0f, __uint_as_float(acc[j]), __shfl_sync(0xffffffffu, hv, j));
                } else {
                    float xv[32];
                    const float cpv = __ldg(args.cprime + i0 + lane);
#pragma unroll
                    for (int j = 0; j < 32; ++j) xv[j] = args.x[(size_t)(i0 + j) * args.B + b];
                    tc_wait_ld();
#pragma unroll
                    for (int j = 0; j < 32; ++j) {                                // x_hat_i ((Q_off x_hat)_i + c'_i), fp32 row sums
                        const float cpj = __shfl_sync(0xffffffffu, cpv, j);
                        if (xv[j] > 0.5f) score += (double)__uint_as_float(acc[j]) + (double)cpj;
                    }
                }
            }
            if (MODE == MODE_SCORE) {                       // one partial per 128 variables
                const int slot = (t.n0 + half * hcols) / 128;
                args.partial[(size_t)slot * args.B + b] = score;
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {                                                      // CG * 8 warps -> accumulator stage free
                if (CG == 1) mbar_arrive(tempty_bar(as)); else mbar_arrive_cluster(map_to_cta(tempty_bar(as), (uint32_t)lead));
            }
        }
        if (STEP && lane == 0) bulk_wait0();                  // this lane's operand stores are complete before the CTA retires
    }
    tc_fence_before();
    if (CSIZE > 1) cluster_sync_all(); else __syncthreads();      // no CTA leaves while its peer may still signal or read it
    if (warp == 2) {
        tc_fence_after();
        if (CG == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
        else asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
    }
}

// fp32 X [n][B] -> bf16 operand [B][n]: centred (x - 1/2) for the step GEMM, or x_hat = [x > 1/2] for scoring
template <int HAT>
__global__ void __launch_bounds__(256)
make_operand_kernel(int n, int B, const float* __restrict__ x, __nv_bfloat16* __restrict__ zt) {
    __shared__ float tile[32][33];
    const int i0 = blockIdx.x * 32, b0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8) tile[r][tx] = x[(size_t)(i0 + r) * B + b0 + tx];
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const float v = tile[tx][r];
        zt[(size_t)(b0 + r) * n + i0 + tx] = __float2bfloat16_rn(HAT ? (v > 0.5f ? 1.0f : 0.0f) : v - 0.5f);
    }
}

// ---- host side ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

gda_status get_encoder(EncodeTiledFn* fn) {
    static EncodeTiledFn cached = nullptr;
    if (!cached) {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult q;
        GDA_CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &q));
        if (q != cudaDriverEntryPointSuccess || !sym) {
            gda_set_error("cuTensorMapEncodeTiled is not available from this driver");
            return GDA_ERR_CUDA;
        }
        cached = reinterpret_cast<EncodeTiledFn>(sym);
    }
    *fn = cached;
    return GDA_OK;
}

// bf16 row-major [rows][cols] (cols contiguous = K), box = box_rows x 64 elements, 128-byte swizzle
gda_status make_tmap(CUtensorMap* map, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    EncodeTiledFn enc;
    GDA_TRY(get_encoder(&enc));
    const cuuint64_t dims[2] = {cols, rows};
    const cuuint64_t strides[1] = {cols * sizeof(__nv_bfloat16)};
    const cuuint32_t box[2] = {(cuuint32_t)BK, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { gda_set_error("cuTensorMapEncodeTiled failed with CUresult %d", (int)r); return GDA_ERR_CUDA; }
    return GDA_OK;
}

struct DenseHost {
    CUtensorMap tmap_q;
    CUtensorMap tmap_z[2];              // operand loads: boxes of 64 rows
    CUtensorMap tmap_zs[2];             // operand stores from the epilogue: boxes of 32 rows (one epilogue warp's restarts)
    const void* z_ptr[2] = {nullptr, nullptr};
    int32_t z_B = 0;
    // co-resident clusters per kernel variant (1 CTA per SM), see configure_variant
    int max_clusters[4 * 2 * 4] = {};
};

// The launch shapes: single CTAs, pairs, two pairs (1 x 2) and four pairs (2 x 2) per cluster.
constexpr int NUM_SHAPES = 4;
constexpr int shape_index(int cg, int pm, int pn) { return cg == 1 ? 0 : pm * pn == 1 ? 1 : pm == 1 ? 2 : 3; }

// One-time setup of a kernel variant on the handle's device: the shared-memory opt-in and the number of co-resident
// clusters (1 CTA per SM).  Done for every variant at create (dense_prepare) -- not lazily at the first launch, which
// is inside a stream capture -- and kept in the handle: per device, no process-wide state.
template <int MODE, int GFUN, int CG, int PM, int PN>
gda_status configure_variant(gda_problem* p) {
    auto kern = dense_gemm_kernel<MODE, GFUN, CG, PM, PN>;
    constexpr int CSIZE = CG * PM * PN;
    GDA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Pipe<CG>::SMEM_BYTES));
    int max_clusters = p->num_sms / CSIZE;
    if (CSIZE > 2) {                                          // clusters of 4 or 8 do not pack all 148 SMs
        cudaLaunchConfig_t cfg = {};
        cfg.blockDim = dim3(NUM_THREADS); cfg.dynamicSmemBytes = Pipe<CG>::SMEM_BYTES;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = CSIZE; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        cfg.gridDim = dim3((unsigned)(max_clusters * CSIZE));
        int q = 0;
        GDA_CUDA_TRY(cudaOccupancyMaxActiveClusters(&q, kern, &cfg));
        if (q > 0 && q < max_clusters) max_clusters = q;
    }
    static_cast<DenseHost*>(p->tmap_Q)->max_clusters[(MODE * 2 + GFUN) * NUM_SHAPES + shape_index(CG, PM, PN)] = max_clusters;
    return GDA_OK;
}

template <int MODE, int GFUN>
gda_status configure_shapes(gda_problem* p) {
    GDA_TRY((configure_variant<MODE, GFUN, 1, 1, 1>(p)));
    GDA_TRY((configure_variant<MODE, GFUN, 2, 1, 1>(p)));
    GDA_TRY((configure_variant<MODE, GFUN, 2, 1, 2>(p)));
    return configure_variant<MODE, GFUN, 2, 2, 2>(p);
}

gda_status configure_all(gda_problem* p) {
    GDA_TRY((configure_shapes<MODE_STEP, GDA_G_QUADRATIC>(p)));
    GDA_TRY((configure_shapes<MODE_STEP, GDA_G_ENTROPY>(p)));
    GDA_TRY((configure_shapes<MODE_STEP_S, GDA_G_QUADRATIC>(p)));
    GDA_TRY((configure_shapes<MODE_STEP_S, GDA_G_ENTROPY>(p)));
    GDA_TRY((configure_shapes<MODE_GRAD, GDA_G_QUADRATIC>(p)));
    return configure_shapes<MODE_SCORE, GDA_G_QUADRATIC>(p);
}

template <int MODE, int GFUN, int CG, int PM, int PN>
gda_status launch_variant(gda_problem* p, const CUtensorMap& ta, const CUtensorMap& tq, const CUtensorMap& tzo, const DenseArgs& a, cudaStream_t s) {
    auto kern = dense_gemm_kernel<MODE, GFUN, CG, PM, PN>;
    constexpr int CSIZE = CG * PM * PN;
    const int max_clusters = static_cast<DenseHost*>(p->tmap_Q)->max_clusters[(MODE * 2 + GFUN) * NUM_SHAPES + shape_index(CG, PM, PN)];
    if (max_clusters <= 0) { gda_set_error("dense path: kernel variant was not configured at create"); return GDA_ERR_CUDA; }
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(NUM_THREADS); cfg.dynamicSmemBytes = Pipe<CG>::SMEM_BYTES; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CSIZE; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    const int units = (a.B / (BM * CG * PM)) * (a.n / (BN * PN));
    const int rounds = (units + max_clusters - 1) / max_clusters;
    const int clusters = (units + rounds - 1) / rounds;       // fewest clusters that still finish in `rounds` rounds
    cfg.gridDim = dim3((unsigned)(clusters * CSIZE));
    GDA_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, ta, tq, tzo, a));
    return GDA_OK;
}

// GDA_OPT_DENSE_SHAPE = 0..3 forces a launch shape the sizes allow (tests, A/B timing); default: the largest cluster that fits
template <int MODE, int GFUN>
gda_status launch_gemm(gda_problem* p, const CUtensorMap& ta, const CUtensorMap& tzo, const DenseArgs& a, cudaStream_t s) {
    DenseHost* h = static_cast<DenseHost*>(p->tmap_Q);
    int shape = a.B % (BM * 2) != 0 ? 0 : a.n % (BN * 2) != 0 ? 1 : a.B % (BM * 4) != 0 ? 2 : 3;
    if (shape == 3 && p->opt_dense_shape < 0) {
        // Clusters of 8 move a third less operand data per tile (measured on config 4: 30 us per round against 34 us)
        // but only 15 of them are co-resident on a B200 (120 SMs) against 33 clusters of 4: take them only when the
        // round count does not eat the gain (config 4: 64 units -> 5 rounds x 30 us against 4 x 34 us: clusters of 4).
        const int* mc = h->max_clusters + (MODE * 2 + GFUN) * NUM_SHAPES;
        const long units8 = (long)(a.B / (BM * 4)) * (a.n / (BN * 2)), units4 = (long)(a.B / (BM * 2)) * (a.n / (BN * 2));
        const long rounds8 = (units8 + mc[3] - 1) / mc[3], rounds4 = (units4 + mc[2] - 1) / mc[2];
        if (15 * rounds8 >= 17 * rounds4) shape = 2;
    }
    if (p->opt_dense_shape >= 0 && p->opt_dense_shape < shape) shape = p->opt_dense_shape;
    switch (shape) {
        case 0: return launch_variant<MODE, GFUN, 1, 1, 1>(p, ta, h->tmap_q, tzo, a, s);
        case 1: return launch_variant<MODE, GFUN, 2, 1, 1>(p, ta, h->tmap_q, tzo, a, s);
        case 2: return launch_variant<MODE, GFUN, 2, 1, 2>(p, ta, h->tmap_q, tzo, a, s);
        default: return launch_variant<MODE, GFUN, 2, 2, 2>(p, ta, h->tmap_q, tzo, a, s);
    }
}

// the load map of an operand buffer and (store != NULL) its store map
gda_status z_maps(gda_problem* p, int32_t B, const __nv_bfloat16* zt, const CUtensorMap** load, const CUtensorMap** store = nullptr) {
    DenseHost* h = static_cast<DenseHost*>(p->tmap_Q);
    int k = -1;
    for (int q = 0; q < 2; ++q)
        if (h->z_ptr[q] == zt && h->z_B == B) k = q;
    if (k < 0) {
        if (h->z_B != B || (h->z_ptr[0] && h->z_ptr[1])) { h->z_ptr[0] = h->z_ptr[1] = nullptr; h->z_B = B; }   // stale entries
        k = h->z_ptr[0] == nullptr ? 0 : 1;
        GDA_TRY(make_tmap(&h->tmap_z[k], zt, (uint64_t)B, (uint64_t)p->n_pad, BBOX));
        GDA_TRY(make_tmap(&h->tmap_zs[k], zt, (uint64_t)B, (uint64_t)p->n_pad, 32));
        h->z_ptr[k] = zt;
    }
    if (load) *load = &h->tmap_z[k];
    if (store) *store = &h->tmap_zs[k];
    return GDA_OK;
}

}  // namespace

// Ragged sizes are served by ZERO PADDING: n is rounded up to a multiple of 256 and (in the workspace) B to a multiple
// of 128, so the kernels only ever see full tiles.  A padding variable has a zero row and column in Q_off, the start
// value x = 0 and a huge constant gradient (h = c' = 1e30): Eq. 6 keeps it at x = 0 (clip), where g(0) = 0, g'(0) is
// finite, the perturbation band is far away and x_hat = 0 adds nothing to F; its operand entry z = -1/2 multiplies
// zeros.  Padding restarts run like any other and are never read.
gda_status dense_prepare(gda_problem* p, const float* Q, const float* c) {
    const int n = p->n, np = p->n_pad;
    std::vector<__nv_bfloat16> qb((size_t)np * np, __float2bfloat16_rn(0.0f));
    std::vector<float> hvec(np, 1e30f), cp(np, 1e30f);
    for (int i = 0; i < n; ++i) {
        double rs = 0.0;
        for (int j = 0; j < n; ++j) {
            const __nv_bfloat16 v = __float2bfloat16_rn(j == i ? 0.0f : Q[(size_t)i * n + j]);
            qb[(size_t)i * np + j] = v;
            rs += (double)__bfloat162float(v);
        }
        cp[i] = (c ? c[i] : 0.0f) + Q[(size_t)i * n + i];                // fold the diagonal (reading R1)
        hvec[i] = (float)(rs + (double)cp[i]);                          // Q_off 1 + c'
    }
    GDA_CUDA_TRY(cudaMalloc((void**)&p->d_Qbf, qb.size() * sizeof(__nv_bfloat16)));
    GDA_CUDA_TRY(cudaMemcpy(p->d_Qbf, qb.data(), qb.size() * sizeof(__nv_bfloat16), cudaMemcpyHostToDevice));
    GDA_CUDA_TRY(cudaMalloc((void**)&p->d_rowsum, np * sizeof(float)));
    GDA_CUDA_TRY(cudaMemcpy(p->d_rowsum, hvec.data(), np * sizeof(float), cudaMemcpyHostToDevice));
    GDA_CUDA_TRY(cudaMalloc((void**)&p->d_cprime, np * sizeof(float)));
    GDA_CUDA_TRY(cudaMemcpy(p->d_cprime, cp.data(), np * sizeof(float), cudaMemcpyHostToDevice));
    DenseHost* h = new DenseHost();
    p->tmap_Q = h;
    GDA_TRY(configure_all(p));
    return make_tmap(&h->tmap_q, p->d_Qbf, (uint64_t)np, (uint64_t)np, BBOX);
}

void dense_release(gda_problem* p) {
    cudaFree(p->d_Qbf); cudaFree(p->d_rowsum);
    p->d_Qbf = nullptr; p->d_rowsum = nullptr;
    delete static_cast<DenseHost*>(p->tmap_Q);
    p->tmap_Q = nullptr;
}

gda_status dense_make_operand(gda_problem* p, int32_t B, const float* x, __nv_bfloat16* zt, int hat, cudaStream_t s,
                              int64_t* launches) {
    dim3 grid((unsigned)(p->n_pad / 32), (unsigned)(B / 32));
    if (hat) make_operand_kernel<1><<<grid, 256, 0, s>>>(p->n_pad, B, x, zt);
    else make_operand_kernel<0><<<grid, 256, 0, s>>>(p->n_pad, B, x, zt);
    if (launches) ++*launches;
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}

gda_status dense_step(gda_problem* p, int32_t B, float* x, float* y, const __nv_bfloat16* zt_in, __nv_bfloat16* zt_out,
                      const UpdParams& up, const ScalarDual& sd, const RunState* st, uint32_t t_off, cudaStream_t s,
                      int64_t* launches) {
    const CUtensorMap *ta, *tzo;
    GDA_TRY(z_maps(p, B, zt_in, &ta));
    GDA_TRY(z_maps(p, B, zt_out, nullptr, &tzo));
    GDA_TRY(z_maps(p, B, zt_in, &ta));                        // (a miss on zt_out may have dropped stale entries)
    DenseArgs a{};
    a.n = p->n_pad; a.B = B; a.x = x; a.y = y; a.zt_out = zt_out; a.hvec = p->d_rowsum; a.cprime = p->d_cprime;
    a.up = up; a.st = st; a.t_off = t_off; a.mu = sd.mu; a.gpart = sd.gpart;
    if (launches) ++*launches;
    if (sd.mu) {                                               // PDBO-s
        if (up.gfun == GDA_G_QUADRATIC) return launch_gemm<MODE_STEP_S, GDA_G_QUADRATIC>(p, *ta, *tzo, a, s);
        return launch_gemm<MODE_STEP_S, GDA_G_ENTROPY>(p, *ta, *tzo, a, s);
    }
    if (up.gfun == GDA_G_QUADRATIC) return launch_gemm<MODE_STEP, GDA_G_QUADRATIC>(p, *ta, *tzo, a, s);
    return launch_gemm<MODE_STEP, GDA_G_ENTROPY>(p, *ta, *tzo, a, s);
}

// gda_grad: operand from x (centred), GEMM, G written out.  Uses zt[0] of the workspace as scratch.
gda_status dense_grad(gda_problem* p, int32_t B, const float* x, float* G, cudaStream_t s) {
    Workspace& ws = p->ws;
    ws.has_state = false;                                               // zt[0] is clobbered
    GDA_TRY(dense_make_operand(p, B, x, ws.zt[0], 0, s, nullptr));
    const CUtensorMap* ta;
    GDA_TRY(z_maps(p, B, ws.zt[0], &ta));
    DenseArgs a{};
    a.n = p->n_pad; a.B = B; a.hvec = p->d_rowsum; a.cprime = p->d_cprime; a.gout = G;
    return launch_gemm<MODE_GRAD, GDA_G_QUADRATIC>(p, *ta, *ta, a, s);
}

int32_t dense_num_partials(const gda_problem* p, int32_t) { return p->n_pad / 128; }

// S5: x_hat operand (exact in bf16), GEMM, per-thread column sums.  Scratch: the zt buffer NOT holding the current operand.
gda_status dense_score_partials(gda_problem* p, int32_t B, const float* x, void* partial, int32_t* n_part,
                                cudaStream_t s, int64_t* launches) {
    Workspace& ws = p->ws;
    __nv_bfloat16* scratch = ws.zt[ws.score_scratch];
    GDA_TRY(dense_make_operand(p, B, x, scratch, 1, s, launches));
    const CUtensorMap* ta;
    GDA_TRY(z_maps(p, B, scratch, &ta));
    DenseArgs a{};
    a.n = p->n_pad; a.B = B; a.x = const_cast<float*>(x); a.hvec = p->d_rowsum; a.cprime = p->d_cprime;
    a.partial = static_cast<double*>(partial);
    *n_part = dense_num_partials(p, B);
    if (launches) ++*launches;
    return launch_gemm<MODE_SCORE, GDA_G_QUADRATIC>(p, *ta, *ta, a, s);
}
