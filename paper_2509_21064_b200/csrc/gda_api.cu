// gda_api.cu -- the C ABI of include/gda.h: validation and preprocessing at create, workspace,
// CUDA-graph-captured run loop, host-buffer variant, single-step entry points.
#include "gda_internal.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

int sparse_heavy_threshold();

// ---------------------------------------------------------------------------------------------------
// errors
// ---------------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

void gda_set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char* gda_last_error(void) { return g_err; }
extern "C" const char* gda_version(void) { return "gda-b200 0.1 (sm_100a)"; }

#define GDA_REQUIRE(cond, ...)                 \
    do {                                       \
        if (!(cond)) {                         \
            gda_set_error(__VA_ARGS__);        \
            return GDA_ERR_INVALID_ARG;        \
        }                                      \
    } while (0)

template <typename T>
static gda_status upload(T** dptr, const std::vector<T>& h) {
    *dptr = nullptr;
    const size_t bytes = std::max<size_t>(h.size(), 1) * sizeof(T);
    if (cudaMalloc((void**)dptr, bytes) != cudaSuccess) {
        gda_set_error("device allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(cudaGetLastError()));
        return GDA_ERR_ALLOC;
    }
    if (!h.empty()) GDA_CUDA_TRY(cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    return GDA_OK;
}

static gda_status device_setup(gda_problem* p) {
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || count == 0) {
        gda_set_error("no usable CUDA device (%s); this library has no CPU fallback",
                      e != cudaSuccess ? cudaGetErrorString(e) : "device count is 0");
        cudaGetLastError();
        return GDA_ERR_CUDA;
    }
    GDA_CUDA_TRY(cudaGetDevice(&p->device));
    cudaDeviceProp prop;
    GDA_CUDA_TRY(cudaGetDeviceProperties(&prop, p->device));
    if (prop.major != 10) {
        gda_set_error("device '%s' is sm_%d%d; this library is built for sm_100a (B200) only", prop.name,
                      prop.major, prop.minor);
        return GDA_ERR_UNSUPPORTED;
    }
    p->num_sms = prop.multiProcessorCount;
    p->l2_bytes = prop.l2CacheSize > 0 ? (int64_t)prop.l2CacheSize : p->l2_bytes;
    return GDA_OK;
}

// Entry points run on the problem's device and leave the caller's current device as they found it.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; cudaGetLastError(); }
        if (prev != dev) err = cudaSetDevice(dev); else prev = -1;            // nothing to restore
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define GDA_ON_DEVICE(p) DeviceGuard dev_guard__((p)->device); GDA_CUDA_TRY(dev_guard__.err)

static bool is_integer_valued(float v, float limit) { return std::isfinite(v) && v == std::nearbyint(v) && std::fabs(v) <= limit; }

// ---------------------------------------------------------------------------------------------------
// create: sparse QUBO
// ---------------------------------------------------------------------------------------------------
// Processing order of the light rows for the warp-per-row step kernel: a block takes 8 consecutive rows of this list, and a
// neighbour that sits in the same block is read by that block anyway (as the neighbour's own x), so its gather is an L1 hit
// instead of another 512 bytes out of the L2 (config 3: L2 -> SM reads 125.6 -> 97.7 MB per step, L1 hit rate 27 -> 41 %).
// Measured: the PDBO step does not get faster (14.95 -> 15.15 us: it is bound by the latency of its dependent loads, not by
// L2 bytes), the PDBO-s step does (20.15 -> 19.2 us: its blocks end in a barrier and wait for their slowest warp), so the
// list is used for PDBO-s only (sparse_step).  Greedy
// growth of groups of 8: start at an unassigned row, keep adding the unassigned neighbour with the most links into the
// group; groups that close early (no unassigned neighbour left) are packed together at the end.  The state arrays keep the
// caller's row order: only WHICH rows share a block changes.  Returns false (and leaves `order` alone) when the list as given
// already has at least as many in-block neighbours, e.g. a banded matrix in its natural order.
static bool locality_order(int n, const std::vector<int32_t>& rowptr, const std::vector<int32_t>& col, const std::vector<int32_t>& rows,
                           std::vector<int32_t>* order) {
    constexpr int K = 8;
    std::vector<uint8_t> taken(n, 1);                         // rows outside the list (row-split kernel) are never grouped
    for (int32_t r : rows) taken[r] = 0;
    std::vector<int32_t> full, frag, group, cand, links(n, 0);
    full.reserve(rows.size());
    for (int32_t seed : rows) {
        if (taken[seed]) continue;
        group.assign(1, seed); cand.clear();
        taken[seed] = 1;
        for (int32_t v = seed; (int)group.size() <= K;) {
            for (int k = rowptr[v]; k < rowptr[v + 1]; ++k) {
                const int32_t j = col[k];
                if (!taken[j] && links[j]++ == 0) cand.push_back(j);
            }
            if ((int)group.size() == K || cand.empty()) break;
            size_t best = 0;
            for (size_t q = 1; q < cand.size(); ++q)
                if (links[cand[q]] > links[cand[best]] || (links[cand[q]] == links[cand[best]] && cand[q] < cand[best])) best = q;
            v = cand[best];
            cand[best] = cand.back(); cand.pop_back();
            links[v] = 0; taken[v] = 1;
            group.push_back(v);
        }
        for (int32_t j : cand) links[j] = 0;
        auto& dst = (int)group.size() == K ? full : frag;
        dst.insert(dst.end(), group.begin(), group.end());
    }
    full.insert(full.end(), frag.begin(), frag.end());
    auto in_block = [&](const std::vector<int32_t>& list) {   // gathers whose target is processed by the same block
        std::vector<int32_t> block_of(n, -1);
        for (size_t q = 0; q < list.size(); ++q) block_of[list[q]] = (int32_t)(q / K);
        int64_t cnt = 0;
        for (int32_t r : list)
            for (int k = rowptr[r]; k < rowptr[r + 1]; ++k) cnt += block_of[col[k]] == block_of[r];
        return cnt;
    };
    if (in_block(full) <= in_block(rows)) return false;
    *order = full;
    return true;
}

extern "C" gda_status gda_create_qubo_csr(int32_t n, const int32_t* rowptr, const int32_t* col, const float* val,
                                          const float* c, gda_problem** out) {
    if (out) *out = nullptr;
    GDA_REQUIRE(out != nullptr, "gda_create_qubo_csr: out is NULL");
    GDA_REQUIRE(n > 0, "gda_create_qubo_csr: n must be > 0 (got %d)", n);
    GDA_REQUIRE(rowptr != nullptr, "gda_create_qubo_csr: rowptr is NULL");
    GDA_REQUIRE(rowptr[0] == 0, "gda_create_qubo_csr: rowptr[0] must be 0");
    for (int i = 0; i < n; ++i)
        GDA_REQUIRE(rowptr[i + 1] >= rowptr[i], "gda_create_qubo_csr: rowptr decreases at row %d", i);
    const int64_t nnz_in = rowptr[n];
    GDA_REQUIRE(nnz_in == 0 || (col != nullptr && val != nullptr), "gda_create_qubo_csr: col/val is NULL");

    // sort each row by column, check range / duplicates / finiteness
    std::vector<std::pair<int32_t, float>> ent((size_t)nnz_in);
    for (int i = 0; i < n; ++i) {
        for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
            GDA_REQUIRE(col[k] >= 0 && col[k] < n, "gda_create_qubo_csr: column %d out of range in row %d", col[k], i);
            GDA_REQUIRE(std::isfinite(val[k]), "gda_create_qubo_csr: non-finite value in row %d", i);
            ent[k] = {col[k], val[k]};
        }
        std::sort(ent.begin() + rowptr[i], ent.begin() + rowptr[i + 1]);
        for (int k = rowptr[i] + 1; k < rowptr[i + 1]; ++k)
            GDA_REQUIRE(ent[k].first != ent[k - 1].first, "gda_create_qubo_csr: duplicate entry (%d,%d)", i, ent[k].first);
    }
    // symmetry: Q_ij == Q_ji exactly
    for (int i = 0; i < n; ++i)
        for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
            const int j = ent[k].first;
            if (j == i) continue;
            auto lo = ent.begin() + rowptr[j], hi = ent.begin() + rowptr[j + 1];
            auto it = std::lower_bound(lo, hi, std::make_pair((int32_t)i, -INFINITY));
            GDA_REQUIRE(it != hi && it->first == i && it->second == ent[k].second,
                        "gda_create_qubo_csr: Q is not symmetric at (%d,%d)", i, j);
        }
    // fold the diagonal into the linear term (reading R1), double the off-diagonal (G = 2 Q_off x + c')
    std::vector<int32_t> h_rowptr(n + 1, 0), h_col;
    std::vector<float> h_val2, h_cp(n);
    std::vector<int32_t> heavy, light;
    h_col.reserve(nnz_in); h_val2.reserve(nnz_in);
    bool integral = true;
    int32_t max_deg = 0;
    for (int i = 0; i < n; ++i) {
        float cp = c ? c[i] : 0.0f;
        GDA_REQUIRE(std::isfinite(cp), "gda_create_qubo_csr: non-finite c[%d]", i);
        double abs_row = 0.0;
        for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
            if (ent[k].first == i) { cp += ent[k].second; continue; }
            h_col.push_back(ent[k].first);
            h_val2.push_back(2.0f * ent[k].second);
            integral = integral && is_integer_valued(ent[k].second, 1048576.0f);
            abs_row += std::fabs(2.0 * ent[k].second);
        }
        h_cp[i] = cp;
        integral = integral && is_integer_valued(cp, 1073741824.0f) && abs_row < 1073741824.0;
        h_rowptr[i + 1] = (int32_t)h_col.size();
        const int32_t deg = h_rowptr[i + 1] - h_rowptr[i];
        max_deg = std::max(max_deg, deg);
        (deg > sparse_heavy_threshold() ? heavy : light).push_back(i);
    }

    gda_problem* p = new (std::nothrow) gda_problem();
    if (!p) { gda_set_error("host allocation failed"); return GDA_ERR_ALLOC; }
    p->kind = GDA_KIND_SPARSE; p->n = n; p->n_pad = n; p->nnz = (int64_t)h_col.size(); p->integral = integral ? 1 : 0;
    p->max_deg = max_deg;
    gda_status st = device_setup(p);
    if (st == GDA_OK) st = sparse_configure(p);
    if (st == GDA_OK) st = upload(&p->d_rowptr, h_rowptr);
    if (st == GDA_OK) st = upload(&p->d_col, h_col);
    if (st == GDA_OK) st = upload(&p->d_val2, h_val2);
    if (st == GDA_OK) st = upload(&p->d_cprime, h_cp);
    if (st == GDA_OK && !heavy.empty()) {
        p->n_heavy = (int32_t)heavy.size(); p->n_light = (int32_t)light.size();
        st = upload(&p->d_heavy_rows, heavy);
        if (st == GDA_OK) st = upload(&p->d_light_rows, light);
    }
    std::vector<int32_t> local;
    if (st == GDA_OK && locality_order(n, h_rowptr, h_col, light, &local)) st = upload(&p->d_local_rows, local);
    if (st == GDA_OK) st = sparse_build_slab(p, h_rowptr, h_col, h_val2);
    if (st == GDA_OK && (int64_t)h_col.size() <= 8 * (int64_t)n) {
        // packed records for rows of degree <= 8 (one 64-byte load replaces rowptr -> col/val): 8 columns then 8
        // values, zeros dropped, padding = (own row, 0); word 0 = -1 sends the row to the CSR path.
        std::vector<int32_t> ell((size_t)n * 16);
        for (int i = 0; i < n; ++i) {
            int32_t* rec = ell.data() + (size_t)i * 16;
            const int32_t deg = h_rowptr[i + 1] - h_rowptr[i];
            for (int q = 0; q < 8; ++q) { rec[q] = i; rec[8 + q] = 0; }
            if (deg > 8) { rec[0] = -1; continue; }
            int cnt = 0;
            for (int k = h_rowptr[i]; k < h_rowptr[i + 1]; ++k) {
                if (h_val2[k] == 0.0f) continue;
                rec[cnt] = h_col[k];
                std::memcpy(&rec[8 + cnt], &h_val2[k], 4);
                ++cnt;
            }
        }
        st = upload(&p->d_ell, ell);
    }
    if (st != GDA_OK) { gda_destroy(p); return st; }
    *out = p;
    return GDA_OK;
}

// ---------------------------------------------------------------------------------------------------
// create: Max-k-Cut -- the same symmetric CSR (validated, sorted, doubled) as the sparse QUBO with c = 0
// ---------------------------------------------------------------------------------------------------
extern "C" gda_status gda_create_maxkcut(int32_t n, int32_t k, const int32_t* rowptr, const int32_t* col, const float* val,
                                         gda_problem** out) {
    if (out) *out = nullptr;
    GDA_REQUIRE(out != nullptr, "gda_create_maxkcut: out is NULL");
    GDA_REQUIRE(k >= 2 && k <= 8, "gda_create_maxkcut: k must be in [2, 8] (got %d)", k);
    GDA_REQUIRE(n > 0 && rowptr != nullptr, "gda_create_maxkcut: n must be > 0 and rowptr non-NULL");
    // the CSR is validated in full by gda_create_qubo_csr below; what the diagonal scan itself reads is checked first
    GDA_REQUIRE(rowptr[0] == 0, "gda_create_maxkcut: rowptr[0] must be 0");
    for (int i = 0; i < n; ++i)
        GDA_REQUIRE(rowptr[i + 1] >= rowptr[i], "gda_create_maxkcut: rowptr decreases at row %d", i);
    GDA_REQUIRE(rowptr[n] == 0 || (col != nullptr && val != nullptr), "gda_create_maxkcut: col/val is NULL");
    for (int i = 0; i < n; ++i)
        for (int a = rowptr[i]; a < rowptr[i + 1]; ++a)
            GDA_REQUIRE(col[a] != i || val[a] == 0.0f, "gda_create_maxkcut: non-zero diagonal entry at node %d", i);
    gda_problem* p = nullptr;
    GDA_TRY(gda_create_qubo_csr(n, rowptr, col, val, nullptr, &p));
    p->kind = GDA_KIND_KCUT;
    p->kparts = k;
    *out = p;
    return GDA_OK;
}

// ---------------------------------------------------------------------------------------------------
// create: dense QUBO (the heavy lifting is in gda_dense.cu)
// ---------------------------------------------------------------------------------------------------
extern "C" gda_status gda_create_qubo_dense(int32_t n, const float* Q, const float* c, int32_t flags,
                                            gda_problem** out) {
    if (out) *out = nullptr;
    GDA_REQUIRE(out != nullptr, "gda_create_qubo_dense: out is NULL");
    GDA_REQUIRE(n > 0, "gda_create_qubo_dense: n must be > 0 (got %d)", n);
    GDA_REQUIRE(Q != nullptr, "gda_create_qubo_dense: Q is NULL");
    if (!(flags & GDA_DENSE_BF16)) { gda_set_error("gda_create_qubo_dense: only GDA_DENSE_BF16 is implemented"); return GDA_ERR_UNSUPPORTED; }
    for (int i = 0; i < n; ++i) {
        GDA_REQUIRE(!c || std::isfinite(c[i]), "gda_create_qubo_dense: non-finite c[%d]", i);
        for (int j = i; j < n; ++j) {
            const float a = Q[(size_t)i * n + j], b = Q[(size_t)j * n + i];
            GDA_REQUIRE(std::isfinite(a), "gda_create_qubo_dense: non-finite Q[%d][%d]", i, j);
            GDA_REQUIRE(a == b, "gda_create_qubo_dense: Q is not symmetric at (%d,%d)", i, j);
        }
    }
    gda_problem* p = new (std::nothrow) gda_problem();
    if (!p) { gda_set_error("host allocation failed"); return GDA_ERR_ALLOC; }
    p->kind = GDA_KIND_DENSE; p->n = n; p->n_pad = (n + 255) / 256 * 256; p->nnz = (int64_t)n * n; p->integral = 0;
    gda_status st = device_setup(p);
    if (st == GDA_OK) st = dense_prepare(p, Q, c);
    if (st != GDA_OK) { gda_destroy(p); return st; }
    *out = p;
    return GDA_OK;
}

// ---------------------------------------------------------------------------------------------------
// create: MaxSAT
// ---------------------------------------------------------------------------------------------------
extern "C" gda_status gda_create_maxsat(int32_t n, int32_t m, const int32_t* cptr, const int32_t* lit, const float* w,
                                        gda_problem** out) {
    if (out) *out = nullptr;
    GDA_REQUIRE(out != nullptr, "gda_create_maxsat: out is NULL");
    GDA_REQUIRE(n > 0 && m > 0, "gda_create_maxsat: n and m must be > 0 (got %d, %d)", n, m);
    GDA_REQUIRE(cptr != nullptr && lit != nullptr, "gda_create_maxsat: cptr/lit is NULL");
    GDA_REQUIRE(cptr[0] == 0, "gda_create_maxsat: cptr[0] must be 0");
    int32_t kmax = 0, kmin = 0x7fffffff;
    bool integral = true;
    std::vector<int32_t> occ(n + 1, 0), tmp;
    for (int j = 0; j < m; ++j) {
        const int k = cptr[j + 1] - cptr[j];
        GDA_REQUIRE(k > 0, "gda_create_maxsat: clause %d is empty", j);
        kmax = std::max(kmax, k);
        kmin = std::min(kmin, k);
        tmp.clear();
        for (int a = cptr[j]; a < cptr[j + 1]; ++a) {
            const int l = lit[a];
            const int v = (l > 0 ? l : -l) - 1;
            GDA_REQUIRE(l != 0 && v < n, "gda_create_maxsat: literal %d of clause %d out of range", l, j);
            tmp.push_back(v);
            ++occ[v + 1];
        }
        std::sort(tmp.begin(), tmp.end());
        for (size_t a = 1; a < tmp.size(); ++a)
            GDA_REQUIRE(tmp[a] != tmp[a - 1], "gda_create_maxsat: variable %d repeated in clause %d", tmp[a], j);
        const float wj = w ? w[j] : 1.0f;
        GDA_REQUIRE(std::isfinite(wj), "gda_create_maxsat: weight of clause %d is non-finite", j);   // any sign: a polynomial in literal-product form
        integral = integral && is_integer_valued(wj, 1048576.0f);
    }
    if (kmax > 65) { gda_set_error("gda_create_maxsat: clauses longer than 65 literals are not supported (got %d)", kmax); return GDA_ERR_UNSUPPORTED; }
    const int64_t L = cptr[m];
    const int32_t kw = std::max(kmax - 1, 1);
    for (int i = 0; i < n; ++i) occ[i + 1] += occ[i];
    std::vector<int32_t> h_vptr(occ), next(occ.begin(), occ.end() - 1);
    std::vector<float> h_coef((size_t)L), h_w(m);
    std::vector<int32_t> h_others((size_t)L * kw, 0x7FFFFFFF);      // ENC_PAD
    for (int j = 0; j < m; ++j) {
        const float wj = w ? w[j] : 1.0f;
        h_w[j] = wj;
        for (int a = cptr[j]; a < cptr[j + 1]; ++a) {
            const int l = lit[a];
            const int v = (l > 0 ? l : -l) - 1;
            const int s = next[v]++;
            h_coef[s] = l > 0 ? -wj : wj;                    // d/dx of p: -1 for a positive literal, +1 for a negated one
            int q = 0;
            for (int b = cptr[j]; b < cptr[j + 1]; ++b)
                if (b != a) {                                  // enc = var | (positive literal ? 0x80000000 : 0)
                    const int lb = lit[b];
                    const uint32_t vb = (uint32_t)((lb > 0 ? lb : -lb) - 1);
                    h_others[(size_t)s * kw + q++] = (int32_t)(vb | (lb > 0 ? 0x80000000u : 0u));
                }
        }
    }
    gda_problem* p = new (std::nothrow) gda_problem();
    if (!p) { gda_set_error("host allocation failed"); return GDA_ERR_ALLOC; }
    p->kind = GDA_KIND_MAXSAT; p->n = n; p->n_pad = n; p->m = m; p->nnz = L; p->integral = integral ? 1 : 0;
    p->kw = kw; p->kmax = kmax; p->kmin = kmin;
    gda_status st = device_setup(p);
    if (st == GDA_OK) st = upload(&p->d_vptr, h_vptr);
    if (st == GDA_OK) st = upload(&p->d_coef, h_coef);
    if (st == GDA_OK) st = upload(&p->d_others, h_others);
    if (st == GDA_OK) st = upload(&p->d_cptr, std::vector<int32_t>(cptr, cptr + m + 1));
    if (st == GDA_OK) st = upload(&p->d_lit, std::vector<int32_t>(lit, lit + L));
    if (st == GDA_OK) st = upload(&p->d_w, h_w);
    if (st != GDA_OK) { gda_destroy(p); return st; }
    *out = p;
    return GDA_OK;
}

// ---------------------------------------------------------------------------------------------------
// workspace / destroy
// ---------------------------------------------------------------------------------------------------
// Wait for the work this handle has enqueued.  NOT cudaDeviceSynchronize: that call is refused -- and invalidates the
// capture -- while ANY stream of the device is capturing, e.g. another handle's first run on another host thread.
static void wait_for_handle(gda_problem* p) {
    if (p->ev_last) cudaEventSynchronize(p->ev_last);
    if (p->own_stream) cudaStreamSynchronize(p->own_stream);
    cudaGetLastError();
}

// records "everything this handle has enqueued so far" (on the caller's stream, after the join)
static gda_status mark_enqueued(gda_problem* p, cudaStream_t user) {
    if (!p->ev_last) GDA_CUDA_TRY(cudaEventCreateWithFlags(&p->ev_last, cudaEventDisableTiming));
    GDA_CUDA_TRY(cudaEventRecord(p->ev_last, user));
    return GDA_OK;
}

static void drop_graphs(gda_problem* p) {
    for (auto& g : p->graphs) {
        if (g.exec) cudaGraphExecDestroy(g.exec);
        if (g.graph) cudaGraphDestroy(g.graph);
    }
    p->graphs.clear();
}

static void free_workspace(gda_problem* p) {
    Workspace& ws = p->ws;
    drop_graphs(p);
    cudaFree(ws.x[0]); cudaFree(ws.x[1]); cudaFree(ws.y); cudaFree(ws.x_bin); cudaFree(ws.best_obj);
    cudaFree(ws.obj_now); cudaFree(ws.improved); cudaFree(ws.partial); cudaFree(ws.state);
    cudaFree(ws.best_restart); cudaFree(ws.best_val); cudaFree(ws.trace_best); cudaFree(ws.trace_ns);
    cudaFree(ws.zt[0]); cudaFree(ws.zt[1]); cudaFree(ws.z); cudaFree(ws.lab);
    cudaFree(ws.mu[0]); cudaFree(ws.mu[1]); cudaFree(ws.gpart); cudaFree(ws.block_min); cudaFree(ws.gacc);
    ws = Workspace();
}

extern "C" void gda_destroy(gda_problem* p) {
    if (!p) return;
    DeviceGuard guard(p->device);
    wait_for_handle(p);
    free_workspace(p);
    cudaFree(p->d_rowptr); cudaFree(p->d_col); cudaFree(p->d_val2); cudaFree(p->d_cprime);
    cudaFree(p->d_heavy_rows); cudaFree(p->d_light_rows); cudaFree(p->d_local_rows); cudaFree(p->d_ell);
    cudaFree(p->d_slab_ent); cudaFree(p->d_slab_goff); cudaFree(p->d_slab_grow); cudaFree(p->d_slab_ent16);
    cudaFree(p->d_vptr); cudaFree(p->d_coef); cudaFree(p->d_others); cudaFree(p->d_cptr); cudaFree(p->d_lit); cudaFree(p->d_w);
    dense_release(p);
    if (p->own_stream) cudaStreamDestroy(p->own_stream);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->ev_last) cudaEventDestroy(p->ev_last);
    cudaGetLastError();
    delete p;
}

static int32_t num_partials(const gda_problem* p, int32_t B) {
    switch (p->kind) {
        case GDA_KIND_SPARSE: return sparse_num_partials(p, B);
        case GDA_KIND_MAXSAT: return maxsat_num_partials(p, B);
        case GDA_KIND_KCUT: return kcut_num_partials(p, B);
        default: return dense_num_partials(p, B);
    }
}

template <typename T>
static gda_status dmalloc(T** ptr, size_t count) {
    const size_t bytes = std::max<size_t>(count, 1) * sizeof(T);
    if (cudaMalloc((void**)ptr, bytes) != cudaSuccess) {
        *ptr = nullptr;
        gda_set_error("device allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(cudaGetLastError()));
        return GDA_ERR_ALLOC;
    }
    return GDA_OK;
}

static const int32_t TRACE_CAP = 4096;

// Row stride of the state arrays: the kernels work on float4s of restarts (dense: on 128-restart tiles), so any B >= 1 is served
// by zero-initialised PADDING RESTARTS up to the next multiple of 4 (128).  They run like any other restart and are never read:
// the evaluation, the trace, the arg-best and the copies out see the first B columns.
// Few restarts (B <= 64) on problems whose step is dominated by gathers (eight or more per row): a multiple of 8 instead, when
// that needs no more lanes per row than the multiple of 4 does (lanes per row = the power of two >= ld / 4).  Rows of x are then
// whole 32-byte sectors and a gather of 10 or 12 restarts reads two sectors instead of two or three: MIS n = 5e4, d = 100 at
// B = 12 42.4 -> 38.9 us per step, config 5 at B = 10 13.4 -> 13.1 us; with few gathers per row the extra state bytes cost more
// than the alignment gains (MIS d = 3 at B = 10: 4.19 -> 4.30 us), hence the condition.
static int32_t lead_dim(const gda_problem* p, int32_t B) {
    if (p->kind == GDA_KIND_DENSE) return (B + 127) / 128 * 128;
    const int32_t r4 = (B + 3) / 4 * 4, r8 = (B + 7) / 8 * 8;
    auto lanes = [](int32_t ld) { int g = 1; while (4 * g < ld) g <<= 1; return g; };
    const bool gathers_dominate = p->kind == GDA_KIND_MAXSAT ? p->nnz >= 4 * (int64_t)p->n : p->nnz >= 8 * (int64_t)p->n;
    return B <= 64 && gathers_dominate && lanes(r8) == lanes(r4) ? r8 : r4;
}

static gda_status ensure_workspace(gda_problem* p, int32_t B) {
    Workspace& ws = p->ws;
    if (ws.B == B) return GDA_OK;
    wait_for_handle(p);
    free_workspace(p);
    const int32_t ld = lead_dim(p, B);                                            // dense: full 128-restart tiles
    const size_t elems = (size_t)p->n_pad * ld;
    const size_t xelems = p->kind == GDA_KIND_KCUT ? elems * p->kparts : elems;   // Max-k-Cut: k planes
    gda_status st = GDA_OK;
    if (p->kind != GDA_KIND_DENSE) {
        if (st == GDA_OK) st = dmalloc(&ws.x[1], xelems);
    } else {
        if (st == GDA_OK) st = dmalloc(&ws.zt[0], elems);
        if (st == GDA_OK) st = dmalloc(&ws.zt[1], elems);
    }
    if (p->kind == GDA_KIND_KCUT) {
        if (st == GDA_OK) st = dmalloc(&ws.z, xelems);
        if (st == GDA_OK) st = dmalloc(&ws.lab, elems);
    }
    if (st == GDA_OK) st = dmalloc(&ws.x[0], xelems);
    if (st == GDA_OK) st = dmalloc(&ws.y, elems);
    if (st == GDA_OK) st = dmalloc(&ws.x_bin, elems);
    if (st == GDA_OK) st = dmalloc(&ws.best_obj, (size_t)ld);
    if (st == GDA_OK) st = dmalloc(&ws.obj_now, (size_t)ld);
    if (st == GDA_OK) st = dmalloc(&ws.improved, (size_t)ld);
    ws.B = B; ws.ld = ld;                                      // the partial counts below depend on them
    ws.n_part = num_partials(p, ld);
    // + room for the y g(x) partial rows of gda_lagrangian
    if (st == GDA_OK) st = dmalloc((double**)&ws.partial, ((size_t)ws.n_part + (size_t)(p->n_pad + 63) / 64 * 2) * ld);
    if (p->kind != GDA_KIND_KCUT) {                           // PDBO-s state (a few rows of B floats)
        ws.n_gpart = p->kind == GDA_KIND_DENSE ? p->n_pad / 128 : p->kind == GDA_KIND_MAXSAT ? maxsat_num_gparts(p) : 0;
        if (st == GDA_OK) st = dmalloc(&ws.mu[0], (size_t)ld);
        if (st == GDA_OK) st = dmalloc(&ws.mu[1], (size_t)ld);
        if (st == GDA_OK) st = dmalloc(&ws.gpart, (size_t)ws.n_gpart * ld);
        if (st == GDA_OK && p->kind == GDA_KIND_SPARSE) st = dmalloc(&ws.gacc, 2 * (size_t)GDA_GACC_WAYS * ld);   // S^t and S^{t+1}, by the parity of x
    }
    if (st == GDA_OK) st = dmalloc(&ws.state, 1);
    if (st == GDA_OK) st = dmalloc(&ws.block_min, (size_t)(ld + 7) / 8);          // one per block of finalize_kernel (32 restarts) or of the slab kernel (8)
    if (st == GDA_OK) st = dmalloc(&ws.best_restart, 1);
    if (st == GDA_OK) st = dmalloc(&ws.best_val, 1);
    ws.trace_cap = TRACE_CAP;
    if (st == GDA_OK) st = dmalloc(&ws.trace_best, (size_t)TRACE_CAP);
    if (st == GDA_OK) st = dmalloc(&ws.trace_ns, (size_t)TRACE_CAP);
    if (st != GDA_OK) { free_workspace(p); return st; }
    return GDA_OK;
}

// [rows][ld] in the workspace -> [rows][B] at the caller (host or device)
static gda_status copy_out(void* dst, size_t B, const void* src, size_t ld, size_t rows, size_t esz, cudaStream_t s) {
    if (ld == B) GDA_CUDA_TRY(cudaMemcpyAsync(dst, src, rows * B * esz, cudaMemcpyDefault, s));
    else GDA_CUDA_TRY(cudaMemcpy2DAsync(dst, B * esz, src, ld * esz, B * esz, rows, cudaMemcpyDefault, s));
    return GDA_OK;
}
static gda_status copy_in(void* dst, size_t ld, const void* src, size_t B, size_t rows, size_t esz, cudaStream_t s) {
    if (ld == B) GDA_CUDA_TRY(cudaMemcpyAsync(dst, src, rows * B * esz, cudaMemcpyDefault, s));
    else GDA_CUDA_TRY(cudaMemcpy2DAsync(dst, ld * esz, src, B * esz, B * esz, rows, cudaMemcpyDefault, s));
    return GDA_OK;
}

// the caller's stream, or our own when the caller's cannot be captured (legacy default stream)
static gda_status pick_stream(gda_problem* p, void* stream, cudaStream_t* user, cudaStream_t* exec) {
    *user = (cudaStream_t)stream;
    if (stream != nullptr && *user != cudaStreamLegacy) { *exec = *user; return GDA_OK; }
    if (!p->own_stream) {
        GDA_CUDA_TRY(cudaStreamCreateWithFlags(&p->own_stream, cudaStreamNonBlocking));
        GDA_CUDA_TRY(cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming));
        GDA_CUDA_TRY(cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming));
    }
    *exec = p->own_stream;
    GDA_CUDA_TRY(cudaEventRecord(p->ev_fork, *user));
    GDA_CUDA_TRY(cudaStreamWaitEvent(*exec, p->ev_fork, 0));
    return GDA_OK;
}

static gda_status join_stream(gda_problem* p, cudaStream_t user, cudaStream_t exec) {
    if (user != exec) {
        GDA_CUDA_TRY(cudaEventRecord(p->ev_join, exec));
        GDA_CUDA_TRY(cudaStreamWaitEvent(user, p->ev_join, 0));
    }
    return mark_enqueued(p, user);
}

// ---------------------------------------------------------------------------------------------------
// one chunk = `len` GDA steps followed by one evaluation (round, score, best-so-far, commit)
// ---------------------------------------------------------------------------------------------------
static UpdParams make_upd(const gda_params& prm) {
    UpdParams up;
    up.alpha = prm.alpha; up.beta = prm.beta; up.delta = prm.delta; up.log_eps = prm.log_eps;
    up.gfun = prm.gfun;
    up.seed_mix = mix32((uint32_t)prm.seed ^ ((uint32_t)(prm.seed >> 32) * 0x9E3779B9u));
    return up;
}

static gda_status enqueue_chunk(gda_problem* p, int32_t B, int32_t len, int32_t parity, const gda_params& prm,
                                cudaStream_t s, int64_t* launches, int64_t* step_launches) {
    Workspace& ws = p->ws;
    const UpdParams up = make_upd(prm);
    int cur = parity;
    const bool scalar = prm.dual == GDA_DUAL_SCALAR;
    if (p->kind == GDA_KIND_SPARSE) {                         // small n: steps AND evaluation in one launch, state on chip
        int slab = 0;
        const int64_t before = *launches;
        GDA_TRY(sparse_chunk_slab(p, B, ws.ld, len, ws.x[cur], ws.x[cur ^ (len & 1)], ws.y, scalar ? ws.mu[cur] : nullptr,
                                  scalar ? ws.mu[cur ^ (len & 1)] : nullptr, up, s, launches, &slab));   // buffer parity as the per-step kernels leave it
        if (slab) { *step_launches += *launches - before; return GDA_OK; }
    }
    for (int k = 0; k < len; ++k) {
        int64_t before = *launches;
        ScalarDual sd;                                        // PDBO-s: mu follows the parity of x
        if (scalar) {
            sd.mu = ws.mu[cur]; sd.mu_out = ws.mu[cur ^ 1]; sd.gpart = ws.gpart; sd.B = ws.ld; sd.beta = prm.beta; sd.advance = 1;
            if (ws.gacc) {                                    // sparse path: S^t by the parity of x^t, S^{t+1} into the other half
                const size_t half = (size_t)GDA_GACC_WAYS * ws.ld;
                sd.gacc = ws.gacc + (size_t)cur * half; sd.gacc_next = ws.gacc + (size_t)(cur ^ 1) * half;
            }
        }
        if (p->kind == GDA_KIND_SPARSE)
            GDA_TRY(sparse_step(p, ws.ld, ws.x[cur], ws.y, ws.x[cur ^ 1], up, sd, ws.state, (uint32_t)k, s, launches));
        else if (p->kind == GDA_KIND_MAXSAT)
            GDA_TRY(maxsat_step(p, ws.ld, ws.x[cur], ws.y, ws.x[cur ^ 1], up, sd, ws.state, (uint32_t)k, s, launches));
        else if (p->kind == GDA_KIND_KCUT)
            GDA_TRY(kcut_step(p, ws.ld, ws.x[cur], ws.z, ws.y, ws.x[cur ^ 1], up, s, launches));
        else
            GDA_TRY(dense_step(p, ws.ld, ws.x[0], ws.y, ws.zt[cur], ws.zt[cur ^ 1], up, sd, ws.state, (uint32_t)k, s, launches));
        if (scalar && p->kind != GDA_KIND_SPARSE)
            GDA_TRY(gsum_reduce(ws.ld, ws.gpart, ws.n_gpart, prm.beta, ws.mu[cur], ws.mu[cur ^ 1], s, launches));
        *step_launches += *launches - before;
        cur ^= 1;
    }
    const float* xcur = (p->kind == GDA_KIND_DENSE) ? ws.x[0] : ws.x[cur];
    int32_t n_part = 0;
    if (p->kind == GDA_KIND_SPARSE) GDA_TRY(sparse_score_partials(p, ws.ld, xcur, ws.partial, &n_part, s, launches));
    else if (p->kind == GDA_KIND_MAXSAT) GDA_TRY(maxsat_score_partials(p, ws.ld, xcur, ws.partial, &n_part, s, launches));
    else if (p->kind == GDA_KIND_KCUT) GDA_TRY(kcut_score_partials(p, ws.ld, ws.z, ws.lab, ws.partial, &n_part, s, launches));
    else { ws.score_scratch = cur ^ 1; GDA_TRY(dense_score_partials(p, ws.ld, xcur, ws.partial, &n_part, s, launches)); }
    GDA_TRY(eval_finalize(p, B, ws.ld, ws.partial, n_part, ws.obj_now, ws.best_obj, ws.improved, ws.state, ws.trace_best,
                          ws.trace_ns, ws.trace_cap, (uint32_t)len, s, launches));
    if (p->kind == GDA_KIND_KCUT) GDA_TRY(kcut_commit(p, ws.ld, ws.lab, ws.improved, ws.x_bin, s, launches));
    else GDA_TRY(eval_commit(p, ws.ld, xcur, ws.improved, ws.x_bin, s, launches));
    return GDA_OK;
}

// Keys are compared bitwise on canonicalised parameters (canonical_params): fields the kernels ignore are zeroed, so an
// uninitialised or NaN log_eps with the quadratic g cannot force a re-capture on every chunk.
bool GraphKey::operator==(const GraphKey& o) const {
    return B == o.B && len == o.len && parity == o.parity && with_eval == o.with_eval &&
           std::memcmp(&prm.alpha, &o.prm.alpha, sizeof(float)) == 0 && std::memcmp(&prm.beta, &o.prm.beta, sizeof(float)) == 0 &&
           std::memcmp(&prm.delta, &o.prm.delta, sizeof(float)) == 0 && std::memcmp(&prm.log_eps, &o.prm.log_eps, sizeof(float)) == 0 &&
           prm.gfun == o.prm.gfun && prm.seed == o.prm.seed && prm.dual == o.prm.dual;
}

static gda_params canonical_params(const gda_problem* p, const gda_params& in) {
    gda_params c = in;
    if (c.gfun == GDA_G_QUADRATIC) c.log_eps = 0.0f;          // ignored by the quadratic g
    if (p->kind == GDA_KIND_KCUT) c.delta = 0.0f;             // no perturbation for Max-k-Cut (reading K3)
    c.iters = 0; c.eval_every = 0; c.t0 = 0; c.reserved = 0;  // not part of a chunk's identity
    return c;
}

static gda_status launch_chunk(gda_problem* p, int32_t B, int32_t len, int32_t parity, const gda_params& prm,
                               cudaStream_t s) {
    if (!p->opt_graphs || len == 0) {                         // GDA_OPT_GRAPHS
        return enqueue_chunk(p, B, len, parity, prm, s, &p->last_launches, &p->last_step_launches);
    }
    GraphKey key;
    key.B = B; key.len = len; key.parity = parity; key.with_eval = 1; key.prm = canonical_params(p, prm);
    CachedGraph* hit = nullptr;
    for (auto& g : p->graphs) if (g.key == key) { hit = &g; break; }
    if (!hit) {
        if (p->graphs.size() >= 8) drop_graphs(p);
        CachedGraph g;
        g.key = key;
        GDA_CUDA_TRY(cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
        gda_status st = enqueue_chunk(p, B, len, parity, prm, s, &g.launches, &g.step_launches);
        cudaError_t e = cudaStreamEndCapture(s, &g.graph);
        if (st != GDA_OK) { if (g.graph) cudaGraphDestroy(g.graph); return st; }
        if (e != cudaSuccess) { gda_set_error("cudaStreamEndCapture failed: %s", cudaGetErrorString(e)); return GDA_ERR_CUDA; }
        e = cudaGraphInstantiate(&g.exec, g.graph, 0);
        if (e != cudaSuccess) {
            cudaGraphDestroy(g.graph);
            gda_set_error("cudaGraphInstantiate failed: %s", cudaGetErrorString(e));
            return GDA_ERR_CUDA;
        }
        p->graphs.push_back(g);
        hit = &p->graphs.back();
    }
    GDA_CUDA_TRY(cudaGraphLaunch(hit->exec, s));
    p->last_launches += hit->launches;
    p->last_step_launches += hit->step_launches;
    return GDA_OK;
}

// ---------------------------------------------------------------------------------------------------
// gda_run
// ---------------------------------------------------------------------------------------------------
static gda_status check_run_args(const gda_problem* p, int32_t B, const float* x0, const gda_params* prm,
                                 const void* x_bin, const void* obj, const void* best_restart) {
    GDA_REQUIRE(p != nullptr, "gda_run: problem is NULL");
    GDA_REQUIRE(prm != nullptr, "gda_run: params is NULL");
    GDA_REQUIRE(x_bin != nullptr && obj != nullptr && best_restart != nullptr,
                "gda_run: x_bin, obj and best_restart are required");
    GDA_REQUIRE(x0 != nullptr || (p->ws.has_state && p->ws.B == B),
                "gda_run: x0 is NULL but the handle holds no state of a previous run with B = %d to resume", B);
    GDA_REQUIRE(B > 0, "gda_run: B must be positive (got %d)", B);
    GDA_REQUIRE(std::isfinite(prm->alpha) && prm->alpha > 0.0f, "gda_run: alpha must be > 0");
    GDA_REQUIRE(std::isfinite(prm->beta) && prm->beta >= 0.0f, "gda_run: beta must be >= 0");
    GDA_REQUIRE(prm->delta >= 0.0f && prm->delta < 0.5f, "gda_run: delta must be in [0, 1/2)");
    GDA_REQUIRE(prm->eval_every > 0, "gda_run: eval_every must be > 0");
    GDA_REQUIRE(prm->iters >= 0, "gda_run: iters must be >= 0");
    GDA_REQUIRE(prm->gfun == GDA_G_QUADRATIC || prm->gfun == GDA_G_ENTROPY, "gda_run: unknown gfun %d", prm->gfun);
    if (prm->gfun == GDA_G_ENTROPY)
        GDA_REQUIRE(prm->log_eps > 0.0f && prm->log_eps < 0.5f, "gda_run: log_eps must be in (0, 1/2) for the entropy g");
    GDA_REQUIRE(prm->dual == GDA_DUAL_PER_VARIABLE || prm->dual == GDA_DUAL_SCALAR, "gda_run: unknown dual mode %d", prm->dual);
    GDA_REQUIRE(prm->reserved == 0, "gda_run: params->reserved must be 0");
    GDA_REQUIRE(x0 != nullptr || p->ws.dual == prm->dual, "gda_run: a resumed run must keep the dual mode of the run it continues");
    if (prm->dual == GDA_DUAL_SCALAR && p->kind == GDA_KIND_KCUT) {
        gda_set_error("gda_run: Max-k-Cut problems need GDA_DUAL_PER_VARIABLE");
        return GDA_ERR_UNSUPPORTED;
    }
    if ((int64_t)p->n_pad * (int64_t)lead_dim(p, B) * (p->kind == GDA_KIND_KCUT ? p->kparts : 1) >= ((int64_t)1 << 30)) {
        gda_set_error("gda_run: the padded state, %d rows x %d restarts%s, must stay below 2^30 elements (got %lld for n = %d, B = %d): "
                      "kernels use 32-bit byte offsets into X", p->n_pad, lead_dim(p, B), p->kind == GDA_KIND_KCUT ? " x k parts" : "",
                      (long long)p->n_pad * lead_dim(p, B) * (p->kind == GDA_KIND_KCUT ? p->kparts : 1), p->n, B);
        return GDA_ERR_UNSUPPORTED;
    }
    return GDA_OK;
}

// The run itself.  `host` says where x0, lambda0, x_bin, obj and best_restart live: the copies in and out are
// cudaMemcpyDefault (unified addressing tells host from device), everything between them is the same.
static gda_status run_impl(gda_problem* p, int32_t B, const float* x0, const float* lambda0, float lambda0_scalar,
                           const gda_params* prm, uint8_t* x_bin, double* obj, int32_t* best_restart,
                           const gda_extra* extra, void* stream, bool host) {
    GDA_TRY(check_run_args(p, B, x0, prm, x_bin, obj, best_restart));
    GDA_ON_DEVICE(p);
    GDA_TRY(ensure_workspace(p, B));
    cudaStream_t user, s;
    GDA_TRY(pick_stream(p, stream, &user, &s));
    Workspace& ws = p->ws;
    p->last_launches = 0; p->last_step_launches = 0;

    int parity = 0;
    if (x0) {
        ws.has_state = false;
        ws.dual = prm->dual;
        ws.n_eval_host = 0;
        GDA_TRY(run_init(p, B, x0, lambda0, lambda0_scalar, (uint32_t)prm->t0, s, &p->last_launches));
        if (p->kind == GDA_KIND_DENSE)
            GDA_TRY(dense_make_operand(p, ws.ld, ws.x[0], ws.zt[0], /*hat=*/0, s, &p->last_launches));
        if (p->kind == GDA_KIND_SPARSE && prm->dual == GDA_DUAL_SCALAR)      // S^0 for the pipelined multiplier update (parity 0)
            GDA_TRY(sparse_dual_init(p, ws.ld, ws.x[0], prm->gfun, prm->log_eps, ws.gacc, s, &p->last_launches));
        if (p->kind == GDA_KIND_KCUT)                       // run_init put the logits in z; x[0] = SoftMax(z)
            GDA_TRY(kcut_softmax(p, ws.ld, ws.z, ws.x[0], s, &p->last_launches));
    } else {
        parity = ws.parity;      // resume: iterates, duals, best-so-far and the iteration counter stay as they are
        // ... but the internal trace starts over: this call's evaluations land at entry 0 and are what the caller's trace
        // arrays receive, however many evaluations the runs before it recorded (the buffer holds TRACE_CAP per call)
        GDA_CUDA_TRY(cudaMemsetAsync(&ws.state->n_eval, 0, sizeof(uint32_t), s));
        ws.n_eval_host = 0;
    }
    const int32_t full = prm->iters / prm->eval_every, rem = prm->iters % prm->eval_every;
    const int32_t n_eval = std::max(1, full + (rem > 0 ? 1 : 0)), trace_off = ws.n_eval_host;
    for (int32_t c = 0; c < full; ++c) {
        GDA_TRY(launch_chunk(p, B, prm->eval_every, parity, *prm, s));
        parity ^= (prm->eval_every & 1);
    }
    if (rem > 0) { GDA_TRY(launch_chunk(p, B, rem, parity, *prm, s)); parity ^= (rem & 1); }
    if (prm->iters == 0) GDA_TRY(launch_chunk(p, B, 0, parity, *prm, s));     // evaluate the start point
    GDA_TRY(eval_argbest(B, ws.best_obj, ws.best_restart, ws.best_val, s, &p->last_launches));

    ws.parity = parity;
    ws.has_state = true;
    const float* xfin = (p->kind == GDA_KIND_DENSE) ? ws.x[0] : ws.x[parity];
    const size_t ld = (size_t)ws.ld, n = (size_t)p->n;
    GDA_TRY(copy_out(x_bin, (size_t)B, ws.x_bin, ld, n, 1, s));
    GDA_CUDA_TRY(cudaMemcpyAsync(obj, ws.best_obj, (size_t)B * sizeof(double), cudaMemcpyDefault, s));
    GDA_CUDA_TRY(cudaMemcpyAsync(best_restart, ws.best_restart, sizeof(int32_t), cudaMemcpyDefault, s));
    if (extra) {
        if (extra->x_final && p->kind == GDA_KIND_KCUT)      // the logits Z^T, [k][n][B]
            GDA_TRY(copy_out(extra->x_final, (size_t)B, ws.z, ld, n * (size_t)p->kparts, sizeof(float), s));
        else if (extra->x_final) GDA_TRY(copy_out(extra->x_final, (size_t)B, xfin, ld, n, sizeof(float), s));
        if (extra->lambda_final && prm->dual == GDA_DUAL_SCALAR)          // mu^T, [B]
            GDA_CUDA_TRY(cudaMemcpyAsync(extra->lambda_final, ws.mu[parity], (size_t)B * sizeof(float), cudaMemcpyDeviceToDevice, s));
        else if (extra->lambda_final)
            GDA_TRY(copy_out(extra->lambda_final, (size_t)B, ws.y, ld, n, sizeof(float), s));
        if (extra->ones) GDA_TRY(eval_count_ones(p, B, ws.x_bin, extra->ones, s, &p->last_launches));
        if (extra->best_obj) GDA_CUDA_TRY(cudaMemcpyAsync(extra->best_obj, ws.best_val, sizeof(double), cudaMemcpyDeviceToDevice, s));
        // THIS call's evaluations (the internal trace restarts at every call, resumed or not: trace_off == 0)
        const int32_t cnt = std::min(std::min(n_eval, extra->trace_cap), ws.trace_cap - trace_off);
        if (extra->trace_best && cnt > 0) GDA_CUDA_TRY(cudaMemcpyAsync(extra->trace_best, ws.trace_best + trace_off, (size_t)cnt * sizeof(double), cudaMemcpyDeviceToDevice, s));
        if (extra->trace_ns && cnt > 0) GDA_CUDA_TRY(cudaMemcpyAsync(extra->trace_ns, ws.trace_ns + trace_off, (size_t)cnt * sizeof(uint64_t), cudaMemcpyDeviceToDevice, s));
    }
    ws.n_eval_host = std::min(ws.trace_cap, trace_off + n_eval);
    GDA_TRY(join_stream(p, user, s));
    if (host) GDA_CUDA_TRY(cudaStreamSynchronize(user));     // the HOST results are valid when the call returns
    return GDA_OK;
}

extern "C" gda_status gda_run(gda_problem* p, int32_t B, const float* x0, const float* lambda0, float lambda0_scalar,
                              const gda_params* prm, uint8_t* x_bin, double* obj, int32_t* best_restart,
                              const gda_extra* extra, void* stream) {
    return run_impl(p, B, x0, lambda0, lambda0_scalar, prm, x_bin, obj, best_restart, extra, stream, false);
}

// ---------------------------------------------------------------------------------------------------
// gda_run_host: same run, HOST buffers in and out (the copies are part of the call).  No staging buffers and no
// allocation per call: x0 / lambda0 are copied straight into the workspace and the results straight out of it.
// ---------------------------------------------------------------------------------------------------
extern "C" gda_status gda_run_host(gda_problem* p, int32_t B, const float* x0, const float* lambda0,
                                   float lambda0_scalar, const gda_params* prm, uint8_t* x_bin, double* obj,
                                   int32_t* best_restart, void* stream) {
    GDA_REQUIRE(x0 != nullptr, "gda_run_host: x0 is required");
    return run_impl(p, B, x0, lambda0, lambda0_scalar, prm, x_bin, obj, best_restart, nullptr, stream, true);
}

// ---------------------------------------------------------------------------------------------------
// single steps of the path: gradient (S1/S2/S3) and score (S5)
// ---------------------------------------------------------------------------------------------------
extern "C" gda_status gda_grad(gda_problem* p, int32_t B, const float* x, float* G, void* stream) {
    GDA_REQUIRE(p != nullptr && x != nullptr && G != nullptr, "gda_grad: null argument");
    GDA_REQUIRE(B > 0, "gda_grad: B must be positive (got %d)", B);
    GDA_ON_DEVICE(p);
    cudaStream_t user, s;
    if (p->kind == GDA_KIND_KCUT) {
        // x = the logits Z [k][n][B]; G = grad_Z Tr(X W X^T) at X = SoftMax(Z).  Through the workspace
        // (z, x[0] = SoftMax, x[1] = G): the handle's run state is scratch here
        GDA_TRY(ensure_workspace(p, B));
        GDA_TRY(pick_stream(p, stream, &user, &s));
        Workspace& ws = p->ws;
        ws.has_state = false;
        const size_t rows = (size_t)p->n * p->kparts, ld = (size_t)ws.ld;
        if (ld != (size_t)B) GDA_CUDA_TRY(cudaMemsetAsync(ws.z, 0, rows * ld * sizeof(float), s));
        GDA_TRY(copy_in(ws.z, ld, x, (size_t)B, rows, sizeof(float), s));
        GDA_TRY(kcut_softmax(p, ws.ld, ws.z, ws.x[0], s, nullptr));
        GDA_TRY(kcut_grad(p, ws.ld, ws.x[0], ws.x[1], s));
        GDA_TRY(copy_out(G, (size_t)B, ws.x[1], ld, rows, sizeof(float), s));
        return join_stream(p, user, s);
    }
    const bool staged = p->kind != GDA_KIND_DENSE && lead_dim(p, B) != B;     // B % 4 != 0: through the padded workspace arrays
    if (p->kind == GDA_KIND_DENSE || staged) GDA_TRY(ensure_workspace(p, B));
    GDA_TRY(pick_stream(p, stream, &user, &s));
    if (staged) {
        Workspace& ws = p->ws;                               // the handle's run state is scratch here (has_state = false)
        ws.has_state = false;
        GDA_CUDA_TRY(cudaMemsetAsync(ws.x[0], 0, (size_t)p->n * ws.ld * sizeof(float), s));
        GDA_TRY(copy_in(ws.x[0], (size_t)ws.ld, x, (size_t)B, (size_t)p->n, sizeof(float), s));
        if (p->kind == GDA_KIND_SPARSE) GDA_TRY(sparse_grad(p, ws.ld, ws.x[0], ws.x[1], s));
        else GDA_TRY(maxsat_grad(p, ws.ld, ws.x[0], ws.x[1], s));
        GDA_TRY(copy_out(G, (size_t)B, ws.x[1], (size_t)ws.ld, (size_t)p->n, sizeof(float), s));
    } else if (p->kind == GDA_KIND_SPARSE) GDA_TRY(sparse_grad(p, B, x, G, s));
    else if (p->kind == GDA_KIND_MAXSAT) GDA_TRY(maxsat_grad(p, B, x, G, s));
    else {
        Workspace& ws = p->ws;                               // the handle's run state is scratch here (has_state = false)
        if (ws.ld == B && p->n_pad == p->n) {
            GDA_TRY(dense_grad(p, B, x, G, s));
        } else {                                             // ragged sizes: through the zero-padded workspace arrays
            GDA_CUDA_TRY(cudaMemsetAsync(ws.x[0], 0, (size_t)p->n_pad * ws.ld * sizeof(float), s));
            GDA_TRY(copy_in(ws.x[0], (size_t)ws.ld, x, (size_t)B, (size_t)p->n, sizeof(float), s));
            GDA_TRY(dense_grad(p, ws.ld, ws.x[0], ws.y, s));
            GDA_TRY(copy_out(G, (size_t)B, ws.y, (size_t)ws.ld, (size_t)p->n, sizeof(float), s));
        }
    }
    return join_stream(p, user, s);
}

extern "C" gda_status gda_score(gda_problem* p, int32_t B, const float* x, double* obj, void* stream) {
    GDA_REQUIRE(p != nullptr && x != nullptr && obj != nullptr, "gda_score: null argument");
    GDA_REQUIRE(B > 0, "gda_score: B must be positive (got %d)", B);
    GDA_ON_DEVICE(p);
    GDA_TRY(ensure_workspace(p, B));
    cudaStream_t user, s;
    GDA_TRY(pick_stream(p, stream, &user, &s));
    Workspace& ws = p->ws;
    int32_t n_part = 0;
    if (p->kind != GDA_KIND_DENSE && ws.ld != B) {           // B % 4 != 0: a zero-padded copy at the workspace's row stride
        ws.has_state = false;
        float* dst = p->kind == GDA_KIND_KCUT ? ws.z : ws.x[0];
        const size_t rows = (size_t)p->n * (p->kind == GDA_KIND_KCUT ? p->kparts : 1);
        GDA_CUDA_TRY(cudaMemsetAsync(dst, 0, rows * ws.ld * sizeof(float), s));
        GDA_TRY(copy_in(dst, (size_t)ws.ld, x, (size_t)B, rows, sizeof(float), s));
        x = dst;
    }
    if (p->kind == GDA_KIND_SPARSE) GDA_TRY(sparse_score_partials(p, ws.ld, x, ws.partial, &n_part, s, nullptr));
    else if (p->kind == GDA_KIND_MAXSAT) GDA_TRY(maxsat_score_partials(p, ws.ld, x, ws.partial, &n_part, s, nullptr));
    else if (p->kind == GDA_KIND_KCUT) GDA_TRY(kcut_score_partials(p, ws.ld, x, ws.lab, ws.partial, &n_part, s, nullptr));   // x = logits [k][n][B]
    else {
        ws.has_state = false; ws.score_scratch = 1;
        const float* xs = x;
        if (ws.ld != B || p->n_pad != p->n) {                // ragged sizes: zero-padded copy (x_hat = 0 adds nothing)
            GDA_CUDA_TRY(cudaMemsetAsync(ws.x[0], 0, (size_t)p->n_pad * ws.ld * sizeof(float), s));
            GDA_TRY(copy_in(ws.x[0], (size_t)ws.ld, x, (size_t)B, (size_t)p->n, sizeof(float), s));
            xs = ws.x[0];
        }
        GDA_TRY(dense_score_partials(p, ws.ld, xs, ws.partial, &n_part, s, nullptr));
    }
    GDA_TRY(score_reduce(p, B, ws.ld, ws.partial, n_part, obj, s));
    return join_stream(p, user, s);
}

// Per-handle launch options (tests, A/B timing).  Every choice below is read when a chunk is enqueued, i.e. also when a
// graph is captured, so a change drops the handle's cached graphs: the next chunk is captured with the new choice.
extern "C" gda_status gda_set_option(gda_problem* p, int32_t key, int32_t value) {
    GDA_REQUIRE(p != nullptr, "gda_set_option: null handle");
    int32_t* slot = nullptr;
    int32_t lo = 0, hi = 1;
    switch (key) {
        case GDA_OPT_SPARSE_PATH: slot = &p->slab_mode; lo = 0; hi = 2; break;
        case GDA_OPT_SPLIT_ALL_ROWS: slot = &p->opt_split_all; lo = -1; hi = 1; break;
        case GDA_OPT_NARROW_SPLIT: slot = &p->opt_narrow_split; break;
        case GDA_OPT_MAXSAT_NARROW: slot = &p->opt_maxsat_narrow; break;
        case GDA_OPT_DENSE_SHAPE: slot = &p->opt_dense_shape; lo = -1; hi = 3; break;
        case GDA_OPT_GRAPHS: slot = &p->opt_graphs; break;
        case GDA_OPT_ROW_GROUPING: slot = &p->opt_row_grouping; break;
        default: break;
    }
    GDA_REQUIRE(slot != nullptr, "gda_set_option: unknown option %d", key);
    GDA_REQUIRE(value >= lo && value <= hi, "gda_set_option: option %d takes values in [%d, %d] (got %d)", key, lo, hi, value);
    if (key == GDA_OPT_SPARSE_PATH) value = value == 2 ? -1 : value;      // stored as 1 slab / -1 stream / 0 cost model
    if (*slot != value) {
        *slot = value;
        DeviceGuard guard(p->device);
        drop_graphs(p);
    }
    return GDA_OK;
}

extern "C" gda_status gda_get_info(const gda_problem* p, gda_info* info) {
    GDA_REQUIRE(p != nullptr && info != nullptr, "gda_get_info: null argument");
    info->kind = p->kind; info->n = p->n; info->nnz = p->nnz; info->m = p->m; info->integral = p->integral;
    info->last_run_kernel_launches = p->last_launches;
    info->last_run_step_launches = p->last_step_launches;
    return GDA_OK;
}

extern "C" gda_status gda_lagrangian(gda_problem* p, int32_t B, const float* x, const float* lambda, float lambda_scalar,
                                     int32_t gfun, float log_eps, double* out, void* stream) {
    GDA_REQUIRE(p != nullptr && x != nullptr && out != nullptr, "gda_lagrangian: null argument");
    GDA_REQUIRE(B > 0, "gda_lagrangian: B must be positive (got %d)", B);
    GDA_REQUIRE(gfun == GDA_G_QUADRATIC || gfun == GDA_G_ENTROPY, "gda_lagrangian: unknown gfun %d", gfun);
    if (gfun == GDA_G_ENTROPY) GDA_REQUIRE(log_eps > 0.0f && log_eps < 0.5f, "gda_lagrangian: log_eps must be in (0, 1/2)");
    GDA_ON_DEVICE(p);
    GDA_TRY(ensure_workspace(p, B));
    cudaStream_t user, s;
    GDA_TRY(pick_stream(p, stream, &user, &s));
    Workspace& ws = p->ws;
    double* part = static_cast<double*>(ws.partial);
    int32_t n_f = 0, n_g = 0;
    if (p->kind == GDA_KIND_KCUT) {
        // x = the logits Z [k][n][B], lambda [n][B]: L(SoftMax(Z), y) = Tr(X W X^T) + sum_i y_i g(X_:,i)
        ws.has_state = false;
        const size_t rows = (size_t)p->n * p->kparts, ld = (size_t)ws.ld;
        if (ld != (size_t)B) GDA_CUDA_TRY(cudaMemsetAsync(ws.z, 0, rows * ld * sizeof(float), s));
        GDA_TRY(copy_in(ws.z, ld, x, (size_t)B, rows, sizeof(float), s));
        GDA_TRY(kcut_softmax(p, ws.ld, ws.z, ws.x[0], s, nullptr));
        const float* lam = lambda;
        if (lambda && ld != (size_t)B) {
            GDA_CUDA_TRY(cudaMemsetAsync(ws.y, 0, (size_t)p->n * ld * sizeof(float), s));
            GDA_TRY(copy_in(ws.y, ld, lambda, (size_t)B, (size_t)p->n, sizeof(float), s));
            lam = ws.y;
        }
        GDA_TRY(kcut_value_partials(p, ws.ld, ws.x[0], lam, lambda_scalar, gfun, part, &n_f, s));
        GDA_TRY(eval_sum_partials(B, ws.ld, part, n_f, out, s));
        return join_stream(p, user, s);
    }
    if (p->kind == GDA_KIND_DENSE) {
        // f(x) = sum_i x_i (G_i + c'_i) / 2 with G = grad f(x) from the tcgen05 GEMM (bf16 operand: reading R13); the
        // run state of the handle is scratch here, as for gda_grad
        ws.has_state = false;
        const size_t ld = (size_t)ws.ld;
        GDA_CUDA_TRY(cudaMemsetAsync(ws.x[0], 0, (size_t)p->n_pad * ld * sizeof(float), s));
        GDA_TRY(copy_in(ws.x[0], ld, x, (size_t)B, (size_t)p->n, sizeof(float), s));
        GDA_TRY(dense_grad(p, ws.ld, ws.x[0], ws.y, s));
        GDA_TRY(eval_xg_partials(p, ws.ld, ws.x[0], ws.y, part, &n_f, s));
        const float* lam = lambda;
        if (lambda && ld != (size_t)B) {                     // y at the padded stride: G's buffer is free once eval_xg_partials has run
            GDA_TRY(copy_in(ws.y, ld, lambda, (size_t)B, (size_t)p->n, sizeof(float), s));
            lam = ws.y;
        }
        GDA_TRY(eval_yg_partials(p, p->n, ws.ld, ws.x[0], lam, lambda_scalar, gfun, log_eps, part + (size_t)n_f * ld, &n_g, s));
        GDA_TRY(eval_sum_partials(B, ws.ld, part, n_f + n_g, out, s));
        return join_stream(p, user, s);
    }
    const size_t ld = (size_t)ws.ld;
    if (ld != (size_t)B) {                                   // B % 4 != 0: zero-padded copies at the workspace's row stride
        ws.has_state = false;
        GDA_CUDA_TRY(cudaMemsetAsync(ws.x[0], 0, (size_t)p->n * ld * sizeof(float), s));
        GDA_TRY(copy_in(ws.x[0], ld, x, (size_t)B, (size_t)p->n, sizeof(float), s));
        x = ws.x[0];
        if (lambda) {
            GDA_CUDA_TRY(cudaMemsetAsync(ws.y, 0, (size_t)p->n * ld * sizeof(float), s));
            GDA_TRY(copy_in(ws.y, ld, lambda, (size_t)B, (size_t)p->n, sizeof(float), s));
            lambda = ws.y;
        }
    }
    if (p->kind == GDA_KIND_SPARSE) GDA_TRY(sparse_value_partials(p, ws.ld, x, part, &n_f, s));
    else GDA_TRY(maxsat_value_partials(p, ws.ld, x, part, &n_f, s));
    GDA_TRY(eval_yg_partials(p, p->n, ws.ld, x, lambda, lambda_scalar, gfun, log_eps, part + (size_t)n_f * ld, &n_g, s));
    GDA_TRY(eval_sum_partials(B, ws.ld, part, n_f + n_g, out, s));
    return join_stream(p, user, s);
}
