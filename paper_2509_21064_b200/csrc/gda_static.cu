// gda_static.cu -- gda_score_qubo_csr_static: S5 (round + exact score; F of PAPER.md:20) for callers that
// cannot allocate device memory.
//
// Every other entry point of this library works on a gda_problem handle, and a handle is made of cudaMalloc'd memory: the
// device copy of the problem, the iterates, and the [row blocks][B] table of partial objective sums that the scoring
// kernels leave for the reduction that follows them.  Some hosts of a solver cannot accept that:
//   - a process whose own pool allocator was handed all of the HBM at start-up (an inference server, a simulation with a
//     fixed memory plan): a cudaMalloc from a library either fails or eats into a budget that somebody signed off;
//   - a loop with a latency bound: cudaMalloc and cudaFree may synchronise the whole device, so one call from a plug-in
//     stalls every other stream of the process;
//   - code that is only allowed to touch buffers it has been handed (a sandboxed plug-in, a callback that runs while
//     other threads are in the middle of work that an allocation would disturb).
// For them this file scores rounded points of a QUBO whose CSR the caller ALREADY holds in device memory, and keeps the
// partial-sum table in a fixed array that is part of the library's image instead of the heap:
//
//     g_score_scratch: GDA_STATIC_SCRATCH_BYTES = 4 MiB, file scope, `static __device__ __align__(256)`.
//
// What that costs and implies (also stated in include/gda.h):
//   - every GPU on which this library gets loaded holds those 4 MiB from the load to the end of the process, used or not;
//   - the array bounds the problem: B <= GDA_STATIC_SCORE_MAX_B = 4096 restarts (any n: rows are dealt to at most
//     capacity / B row blocks); anything larger is refused with GDA_ERR_UNSUPPORTED and a message that names the limit;
//   - there is ONE array per GPU, shared by every call from every thread and stream.  Two calls that are in flight on the
//     same GPU at the same time (two streams, or two host threads) overwrite each other's partial sums and both return
//     garbage without any error.  Calls on one stream are ordered and safe.  The array keeps whatever the previous call left
//     in it; nothing in it has to start at zero, because each call writes every entry it later reads (each row block
//     stores its sum for each restart, zero included) -- so there is nothing to clear and no memset between calls.
//   - inside HOST code the name `g_score_scratch` is not a device address (it is the host-side shadow the runtime uses as a
//     look-up key); handing it to a kernel would fault or scribble over unrelated memory.  The device address is fetched
//     with cudaGetSymbolAddress, once per GPU, with that GPU current, by the first call made on that GPU.  That first call
//     therefore does a little more than the later ones (it may also trigger the lazy load of this module, which is when
//     the driver places the array) and should be made during start-up, before any stream capture begins.
// No cudaMalloc, cudaFree, cudaMallocAsync, memory pool or allocating library routine is called here -- only
// cudaGetDevice, cudaGetSymbolAddress, cudaPointerGetAttributes and two kernel launches on the caller's stream.
#include "gda_internal.cuh"

#include <mutex>

namespace {

constexpr size_t SCRATCH_DOUBLES = (size_t)GDA_STATIC_SCRATCH_BYTES / sizeof(double);
constexpr int MAX_DEVICES = 64;
constexpr int SCORE_WARPS = 8;              // score block = 32 restarts x 8 warps, a warp takes every 8th row of the block
constexpr int SUM_SLICES = 8;               // sum block   = 32 restarts x 8 slices of row blocks
constexpr int MIN_ROWS_PER_BLOCK = 8;

static __device__ __align__(256) double g_score_scratch[SCRATCH_DOUBLES];

std::mutex g_addr_mutex;
double* g_scratch_addr[MAX_DEVICES] = {};   // device address of g_score_scratch on GPU d, nullptr = not asked yet

#define GDA_STATIC_REQUIRE(cond, status, ...)   \
    do {                                        \
        if (!(cond)) {                          \
            gda_set_error(__VA_ARGS__);         \
            return (status);                    \
        }                                       \
    } while (0)

// partial[rb][b] = sum over the rows i of row block rb with x_hat_ib = 1 of (c_i + sum_k val_k x_hat_{col_k, b}),
// x_hat = [x > 1/2] (exactly 1/2 rounds to 0, reading R5).  Lane = restart, so a gather of one column entry is one
// coalesced 128-byte line per warp and B needs no alignment.  The structure of a row is fetched 32 entries at a time,
// one per lane, and handed round by shuffles (as spmm_score does); sums are taken in fp64 in the order of the CSR, so
// an instance with integer coefficients is scored exactly.  EVERY (rb, b < B) entry is stored, zero sums included.
__global__ void __launch_bounds__(32 * SCORE_WARPS)
static_score_kernel(int n, int B, int rows_per_block, const int32_t* __restrict__ rowptr,
                    const int32_t* __restrict__ col, const float* __restrict__ val, const float* __restrict__ c,
                    const float* __restrict__ x, double* __restrict__ partial) {
    __shared__ double red[SCORE_WARPS][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.y * 32 + lane;
    const bool active = b < B;
    const int row0 = blockIdx.x * rows_per_block;
    double acc = 0.0;
    for (int r = warp; r < rows_per_block; r += SCORE_WARPS) {
        const int row = row0 + r;
        if (row >= n) break;                                 // warp-uniform
        const int start = __ldg(rowptr + row), end = __ldg(rowptr + row + 1);
        double s = 0.0;
        for (int base = start; base < end; base += 32) {
            const int k = base + lane;
            const int my_c = (k < end) ? __ldg(col + k) : 0;
            const float my_v = (k < end) ? __ldg(val + k) : 0.0f;
            const int cnt = min(32, end - base);
            for (int u = 0; u < cnt; ++u) {
                const int cj = __shfl_sync(0xffffffffu, my_c, u);
                const float vj = __shfl_sync(0xffffffffu, my_v, u);
                if (active && __ldg(x + (size_t)cj * B + b) > 0.5f) s += (double)vj;
            }
        }
        if (active && __ldg(x + (size_t)row * B + b) > 0.5f) acc += s + (c ? (double)__ldg(c + row) : 0.0);
    }
    red[warp][lane] = acc;
    __syncthreads();
    if (warp == 0 && active) {
        double t = red[0][lane];
#pragma unroll
        for (int w = 1; w < SCORE_WARPS; ++w) t += red[w][lane];
        partial[(size_t)blockIdx.x * B + b] = t;
    }
}

// obj[b] = sum_rb partial[rb][b], the slices and then the row blocks of a slice added in index order (deterministic)
__global__ void __launch_bounds__(32 * SUM_SLICES)
static_sum_kernel(int B, int n_blocks, const double* __restrict__ partial, double* __restrict__ obj) {
    __shared__ double red[SUM_SLICES][32];
    const int lane = threadIdx.x & 31, slice = threadIdx.x >> 5;
    const int b = blockIdx.x * 32 + lane;
    double s = 0.0;
    if (b < B)
        for (int q = slice; q < n_blocks; q += SUM_SLICES) s += partial[(size_t)q * B + b];   // plain loads: written by the launch before
    red[slice][lane] = s;
    __syncthreads();
    if (slice == 0 && b < B) {
        double t = red[0][lane];
#pragma unroll
        for (int k = 1; k < SUM_SLICES; ++k) t += red[k][lane];
        obj[b] = t;
    }
}

// Device address of the scratch array on the CURRENT GPU; asked for once per GPU (see the file header).
gda_status scratch_on_current_device(double** out) {
    int dev = -1;
    GDA_CUDA_TRY(cudaGetDevice(&dev));
    GDA_STATIC_REQUIRE(dev >= 0 && dev < MAX_DEVICES, GDA_ERR_UNSUPPORTED,
                       "gda_score_qubo_csr_static: device ordinal %d is beyond the %d this build keeps addresses for", dev, MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_addr_mutex);
    if (g_scratch_addr[dev] == nullptr) {
        void* ptr = nullptr;
        GDA_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_score_scratch));
        GDA_STATIC_REQUIRE(ptr != nullptr, GDA_ERR_CUDA, "gda_score_qubo_csr_static: cudaGetSymbolAddress returned a null address");
        g_scratch_addr[dev] = static_cast<double*>(ptr);
    }
    *out = g_scratch_addr[dev];
    return GDA_OK;
}

// A host pointer passed by mistake would fault inside the kernel (or, on a machine where the GPU can reach host memory,
// be read silently); cudaPointerGetAttributes allocates nothing and tells the two apart.
gda_status require_device_pointer(const void* ptr, const char* what) {
    cudaPointerAttributes attr{};
    GDA_CUDA_TRY(cudaPointerGetAttributes(&attr, ptr));
    GDA_STATIC_REQUIRE(attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged, GDA_ERR_INVALID_ARG,
                       "gda_score_qubo_csr_static: %s must be DEVICE memory (this entry point copies nothing)", what);
    return GDA_OK;
}

}  // namespace

extern "C" gda_status gda_score_qubo_csr_static(int32_t n, const int32_t* rowptr, const int32_t* col, const float* val,
                                                const float* c, int32_t B, const float* x, double* obj, void* stream) {
    GDA_STATIC_REQUIRE(rowptr != nullptr && col != nullptr && val != nullptr && x != nullptr && obj != nullptr,
                       GDA_ERR_INVALID_ARG, "gda_score_qubo_csr_static: null argument (only c may be NULL)");
    GDA_STATIC_REQUIRE(n > 0, GDA_ERR_INVALID_ARG, "gda_score_qubo_csr_static: n must be positive (got %d)", n);
    GDA_STATIC_REQUIRE(B > 0, GDA_ERR_INVALID_ARG, "gda_score_qubo_csr_static: B must be positive (got %d)", B);
    GDA_STATIC_REQUIRE(B <= GDA_STATIC_SCORE_MAX_B, GDA_ERR_UNSUPPORTED,
                       "gda_score_qubo_csr_static: B = %d is beyond GDA_STATIC_SCORE_MAX_B = %d, the most the fixed %d-byte scratch "
                       "array serves; score the restarts in slices of at most %d, or use gda_score on a handle",
                       B, GDA_STATIC_SCORE_MAX_B, GDA_STATIC_SCRATCH_BYTES, GDA_STATIC_SCORE_MAX_B);
    double* scratch = nullptr;
    GDA_TRY(scratch_on_current_device(&scratch));
    GDA_TRY(require_device_pointer(rowptr, "rowptr"));
    GDA_TRY(require_device_pointer(col, "col"));
    GDA_TRY(require_device_pointer(val, "val"));
    if (c) GDA_TRY(require_device_pointer(c, "c"));
    GDA_TRY(require_device_pointer(x, "x"));
    GDA_TRY(require_device_pointer(obj, "obj"));

    // rows are dealt to as many row blocks as the array has room for at this B (at least 128, since B <= 4096)
    const size_t max_blocks = SCRATCH_DOUBLES / (size_t)B;
    int rows_per_block = (int)(((size_t)n + max_blocks - 1) / max_blocks);
    if (rows_per_block < MIN_ROWS_PER_BLOCK) rows_per_block = MIN_ROWS_PER_BLOCK;
    const int n_blocks = (n + rows_per_block - 1) / rows_per_block;
    const unsigned col_blocks = (unsigned)((B + 31) / 32);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    static_score_kernel<<<dim3((unsigned)n_blocks, col_blocks), 32 * SCORE_WARPS, 0, s>>>(n, B, rows_per_block, rowptr, col,
                                                                                         val, c, x, scratch);
    GDA_CUDA_TRY(cudaGetLastError());
    static_sum_kernel<<<col_blocks, 32 * SUM_SLICES, 0, s>>>(B, n_blocks, scratch, obj);
    GDA_CUDA_TRY(cudaGetLastError());
    return GDA_OK;
}
