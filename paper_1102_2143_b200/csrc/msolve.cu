// msolve.cu -- C ABI (include/msolve.h) and host-side driver of the multishift solvers.
//
// The host does three things per solve: copy a ~1.6 KB header (pointers, n, shifts, tol) into the
// handle's device-resident SolveState, launch two init kernels and ONE CUDA graph whose WHILE
// node iterates the captured kernel sequence on the device until the device-side stop test
// clears the condition ("entire solution on the GPU"),
// then read back a ~1.6 KB result block after a single stream synchronisation.
// The kernels live in the other translation units (handle.h lists them).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "handle.h"
#include "tuning.h"
#include "spmv_merge.cuh"      // MergeCfg (tile geometry of the merge-path partition built here)

using namespace msolve;

// ------------------------------------------------------------------------------------- errors
static thread_local char g_err[512] = "";

int msolve::fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call) MSOLVE_CU(call)

int msolve::ensure_smem(const msolve_matrix* A, const void* kernel, int bytes) {
    for (const void* k : A->smem_attr_done) if (k == kernel) return MSOLVE_OK;
    CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    A->smem_attr_done.push_back(kernel);
    return MSOLVE_OK;
}

// the handle's device must be the calling thread's current device (kernels, graphs and the function
// attributes above belong to it)
int msolve::check_device(const msolve_matrix* A, const char* who) {
    int cur = -1;
    CU(cudaGetDevice(&cur));
    if (cur != A->device) return fail(MSOLVE_EINVAL, "%s: the handle lives on device %d, the current device is %d", who, A->device, cur);
    return MSOLVE_OK;
}

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
static bool valid_dtype(int dtype) { return dtype >= MSOLVE_C64 && dtype <= MSOLVE_F64; }
static bool complex_dtype(int dtype) { return dtype == MSOLVE_C64 || dtype == MSOLVE_C128; }
static bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

// (lanes, U) of the TMA-staged vector-CSR kernel for rows of at most `maxlen` non-zeros; false when the rows are
// too long.  16-byte elements: U = 4, 2..16 lanes (rows <= 64).  Smaller elements: U = 4 with 2 or 4 lanes
// for rows <= 16 (the 5-point Poisson matrix: 2 x 4 0.0225 ms, 2 x 8 0.0261 ms), U = 8 with
// 4..16 lanes for rows <= 128.
static bool csr_tile_shape(int dtype, long long maxlen, int* lanes, int* u) {
    if (maxlen <= 0) return false;
    if (dtype == MSOLVE_C128 || maxlen <= 16) {
        *u = 4;
        *lanes = 2;
        while (*lanes * 4 < maxlen) *lanes *= 2;
        return *lanes <= 16;
    }
    *u = 8;
    *lanes = 4;
    while (*lanes * 8 < maxlen) *lanes *= 2;
    return *lanes <= 16;
}

#define DISPATCH_ELEM(dtype, EXPR_C128, EXPR_C64, EXPR_F64, EXPR_F32) \
    ((dtype) == MSOLVE_C128 ? (EXPR_C128) : (dtype) == MSOLVE_C64 ? (EXPR_C64) : (dtype) == MSOLVE_F64 ? (EXPR_F64) : (EXPR_F32))

static int merge_diag(int dtype) {
    return DISPATCH_ELEM(dtype, (MergeCfg<double2, MergeTile<double2>::CAP>::kDiag), (MergeCfg<float2, MergeTile<float2>::CAP>::kDiag),
                         (MergeCfg<double, MergeTile<double>::CAP>::kDiag), (MergeCfg<float, MergeTile<float>::CAP>::kDiag));
}

static const char* kCgmNames[] = {"cgm_pupdate", "spmv_dot", "cgm_scal1", "cgm_update", "cgm_scal2", "cgm_flush"};
static const char* kBiNames[] = {"spmv1_dot", "bi_scal1", "bi_supdate", "spmv2_dots", "bi_scal2", "bi_update", "bi_scal3"};
// CG-M with the deferred update: cgm_update is the r update alone and the body ends with the flush kernel (a no-op
// until the chunk is full or the solve has ended)
static int kernels_per_iter(const msolve_matrix* A, int alg) { return alg == MSOLVE_ALG_CGM ? (defer_len(A, alg) > 0 ? 6 : 5) : 7; }
// kernel launches per iteration body: the merge-path SpMV is two launches (tiles + carry fix-up)
static int launches_per_iter(const msolve_matrix* A, int alg) {
    const int spmvs = alg == MSOLVE_ALG_CGM ? 1 : 2;
    return kernels_per_iter(A, alg) + (spmv_launches(A) - 1) * spmvs;
}

// One kernel of the iteration body.  Used for graph capture, and one-by-one for profiling.
static int launch_body_kernel(const msolve_matrix* A, int alg, int j, cudaStream_t s,
                              cudaGraphConditionalHandle cond, int use_cond) {
    if (alg == MSOLVE_ALG_CGM && j == 1) return launch_spmv<ROLE_CG>(A, s);
    if (alg == MSOLVE_ALG_BICGSTABM && j == 0) return launch_spmv<ROLE_B1>(A, s);
    if (alg == MSOLVE_ALG_BICGSTABM && j == 3) return launch_spmv<ROLE_B2>(A, s);
    return launch_vec_kernel(A, alg, j, s, cond, use_cond);
}

// ------------------------------------------------------------------------------------- graph
static int build_graph(msolve_matrix* A, int alg) {
    LoopGraph& g = A->graphs[alg];
    const int key = A->opt.graph_key();
    const SolveHeader& hh = A->h_stage->h;
    const bool same_x = !A->opt.x_window || (g.xptr == hh.p && g.xptr2 == hh.s);
    if (g.exec && g.key == key && same_x) return MSOLVE_OK;
    if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
    if (g.graph) { cudaGraphDestroy(g.graph); g.graph = nullptr; }
    const int nk = kernels_per_iter(A, alg);
    int lrc = MSOLVE_OK;
    if (A->opt.loop_mode == 0) {
        CU(cudaGraphCreate(&g.graph, 0));
        cudaGraphConditionalHandle cond;
        CU(cudaGraphConditionalHandleCreate(&cond, g.graph, 1, cudaGraphCondAssignDefault));
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = cond;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        cudaGraphNode_t node;
        CU(cudaGraphAddNode(&node, g.graph, nullptr, 0, &np));
        cudaGraph_t body = np.conditional.phGraph_out[0];
        CU(cudaStreamBeginCaptureToGraph(A->capture_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
        for (int j = 0; j < nk && lrc == MSOLVE_OK; ++j) lrc = launch_body_kernel(A, alg, j, A->capture_stream, cond, 1);
        cudaError_t le = cudaGetLastError();
        cudaGraph_t dummy = nullptr;
        CU(cudaStreamEndCapture(A->capture_stream, &dummy));
        if (lrc != MSOLVE_OK) return lrc;
        if (le != cudaSuccess) return fail(MSOLVE_ECUDA, "kernel launch during capture failed: %s", cudaGetErrorString(le));
    } else {
        CU(cudaStreamBeginCapture(A->capture_stream, cudaStreamCaptureModeThreadLocal));
        for (int c = 0; c < kChunk && lrc == MSOLVE_OK; ++c)
            for (int j = 0; j < nk && lrc == MSOLVE_OK; ++j) lrc = launch_body_kernel(A, alg, j, A->capture_stream, 0, 0);
        cudaError_t le = cudaGetLastError();
        CU(cudaStreamEndCapture(A->capture_stream, &g.graph));
        if (lrc != MSOLVE_OK) return lrc;
        if (le != cudaSuccess) return fail(MSOLVE_ECUDA, "kernel launch during capture failed: %s", cudaGetErrorString(le));
    }
    CU(cudaGraphInstantiate(&g.exec, g.graph, 0));
    g.key = key; g.xptr = hh.p; g.xptr2 = hh.s;
    return MSOLVE_OK;
}

// AUTO rule of MSOLVE_CFG_ITER_PATH: one cooperative kernel per solve up to this working set.  Measured per-iteration
// times, graph / one kernel (profiles/r02_sweeps.md): 11 MB 23.6 / 18.2 us, 150 MB 86 / 76 us, 200 MB 71 / 63 us,
// 400 MB 119 / 115 us, 800 MB 218 / 223 us.
constexpr size_t kFusedMaxBytes = (size_t)256 << 20;
// CG-M with the deferred multishift update moves 2.2x fewer bytes per iteration as a graph of kernels: measured
// crossover with the one-kernel path at 100 MB (config 4's operator, 16 shifts: n = 98 304; profiles/r02_sweeps.md section 6)
constexpr size_t kFusedMaxBytesDeferred = (size_t)96 << 20;
// ... and with everything resident in shared memory while it fits there (148 x ~200 KB; resident.cu checks the exact
// per-CTA layout, this bound only saves the host copy of rowptr for matrices that cannot fit)
constexpr size_t kResidentMaxBytes = (size_t)28 << 20;
static size_t matrix_bytes(const msolve_matrix* A) {
    const size_t e = elem_bytes(A->dtype);
    if (A->format == FMT_BSR3) return (size_t)A->dev.nnz * (9 * e + 4) + (size_t)(A->dev.nbrows + 1) * 4;
    if (A->format == FMT_LATTICE) return (size_t)A->dev.nnz * 9 * e;
    return (size_t)A->dev.nnz * (e + 4) + (size_t)(A->dev.n + 1) * 4;
}
// ------------------------------------------------------------------------------------- create
static int create_common(msolve_matrix** out, msolve_matrix* A, cudaStream_t stream) {
    (void)stream;
    CU(cudaGetDevice(&A->device));
    CU(cudaDeviceGetAttribute(&A->num_sms, cudaDevAttrMultiProcessorCount, A->device));
    CU(cudaMalloc((void**)&A->d_state, sizeof(SolveState)));
    CU(cudaMemset(A->d_state, 0, sizeof(SolveState)));
    CU(cudaMallocHost((void**)&A->h_stage, sizeof(SolveHeader) + sizeof(SolveResult)));
    CU(cudaStreamCreateWithFlags(&A->capture_stream, cudaStreamNonBlocking));
    A->dev.mat_keep = 0;
    *out = A;
    return MSOLVE_OK;
}

// Tile table of the TMA-staged BSR3 kernel: consecutive block rows, at most TB rows and 9*TB
// blocks per tile, every tile starting at a block index that is a multiple of 4 (16-byte aligned
// bulk copies for both dtypes).  Falls back to the row kernel when no such partition exists.
static int build_bsr_tiles(msolve_matrix* A) {
    const int TB = A->dtype == MSOLVE_C64 ? BsrTile<float2>::TB : BsrTile<double2>::TB;
    const int maxb = 9 * TB;
    const long long nbr = A->dev.nbrows;
    std::vector<int32_t> rp((size_t)nbr + 1);
    CU(cudaMemcpy(rp.data(), A->dev.rowptr, sizeof(int32_t) * (size_t)(nbr + 1), cudaMemcpyDeviceToHost));
    if (rp[0] != 0) return MSOLVE_OK;  // unusual base: keep the row kernel
    std::vector<int4> tiles;
    long long r = 0;
    while (r < nbr) {
        long long end = r, best = -1;
        while (end < nbr && end - r < TB && rp[end + 1] - rp[r] <= maxb) {
            ++end;
            if (rp[end] % 4 == 0 || end == nbr) best = end;
        }
        if (best <= r) return MSOLVE_OK;  // a row is too dense or alignment impossible: row kernel
        tiles.push_back(make_int4((int)r, (int)best, rp[r], rp[best]));
        r = best;
    }
    CU(cudaMalloc(&A->d_aux, sizeof(int4) * tiles.size()));
    CU(cudaMemcpy(A->d_aux, tiles.data(), sizeof(int4) * tiles.size(), cudaMemcpyHostToDevice));
    A->dev.aux = (const int32_t*)A->d_aux;
    A->dev.aux_count = (int)tiles.size();
    A->kernel = KERNEL_BSR_TMA;
    return MSOLVE_OK;
}


// Merge-path partition (spmv_merge.cuh): the n + nnz merge items (row ends, non-zeros) are cut
// every kDiag items.  Split point on diagonal d: i = number of row ends consumed, found by binary
// search for the first i with rowptr[i+1] > d-i-1; k = d - i.  k is then moved up to the next
// multiple of 4 (16-byte aligned bulk copies for values and indices) and i to the first row not
// yet finished at that k.  Tile t = {i0, i1, k0, k1}: rows i0..i1-1 end inside the tile, row i1
// (if < n) may continue.  Also decides AUTO: merge-path when the row lengths are irregular.
static int build_merge_tiles(msolve_matrix* A, int flags, const std::vector<int32_t>& rp) {
    const bool force = flags != MSOLVE_SPMV_AUTO;      // a kernel was asked for by name: bad input is an error
    const long long n = A->dev.n, nnz = A->dev.nnz;
    if (n == 0) return MSOLVE_OK;
    if (rp[0] != 0 || rp[(size_t)n] != nnz) return force ? fail(MSOLVE_EINVAL, "msolve_create_csr: rowptr[0] != 0 or rowptr[n] != nnz") : MSOLVE_OK;
    long long maxlen = 0;
    for (long long i = 0; i < n; ++i) {
        if (rp[i + 1] < rp[i]) return force ? fail(MSOLVE_EINVAL, "msolve_create_csr: rowptr is not non-decreasing") : MSOLVE_OK;
        maxlen = std::max<long long>(maxlen, rp[i + 1] - rp[i]);
    }
    if (maxlen * n == nnz) {   // constant row length (stencils, lattices): lanes by the BYTES of a row (measured,
        const long long rb = maxlen * (long long)elem_bytes(A->dtype);   // config 4 CSR c64: 4 lanes 0.59 ms, 8 lanes 0.75 ms)
        A->lanes = rb > 768 ? 32 : rb > 320 ? 8 : rb > 96 ? 4 : 2;
    }
    // TMA-staged vector-CSR (spmv_csr_tile.cuh): every row fits LANES * U non-zeros, LANES <= 16.
    // AUTO takes it whenever the rows allow it: it is the faster CSR kernel on every workload
    // with short rows (config 4 as CSR, config 3, the 1000 x 1000 Poisson matrix).
    int tl = 0, tu = 0;
    const bool tile_ok = csr_tile_shape(A->dtype, maxlen, &tl, &tu);
    if (flags == MSOLVE_SPMV_TILE && !tile_ok)
        return fail(MSOLVE_EINVAL, "msolve_create_csr: MSOLVE_SPMV_TILE needs rows of 1..%d non-zeros (longest row: %lld)",
                    A->dtype == MSOLVE_C128 ? 64 : 128, maxlen);
    // small matrices (config 2, N = 12288: 0.0088 vs 0.0090 ms per SpMV, 37.2k vs 40.9k iterations/s)
    // do not fill the ring; they stay with the vector kernel
    if (flags == MSOLVE_SPMV_TILE || (flags == MSOLVE_SPMV_AUTO && tile_ok && n >= 65536)) {
        A->lanes = tl;
        A->tile_u = tu;
        A->kernel = KERNEL_CSR_TILE;
        return MSOLVE_OK;
    }
    if (flags != MSOLVE_SPMV_MERGE) {
        const double mean = (double)nnz / (double)n;
        // Vector kernel unless single rows dwarf the mean (a sub-warp would serialise them): on
        // config 5 (rows 5..200, mean 32) the vector kernel is the faster one on B200 (1.14 vs
        // 1.33 ms complex128, 0.91 vs 0.90 ms complex64, profiles/r01_sweeps.md).
        if ((double)maxlen <= 16.0 * mean + 64.0) return MSOLVE_OK;
    }
    const int D = merge_diag(A->dtype);
    const long long items = n + nnz;
    const long long ntiles = (items + D - 1) / D;
    if (ntiles >= (1ll << 31) - 1) return force ? fail(MSOLVE_EINVAL, "msolve_create_csr: too many tiles") : MSOLVE_OK;
    std::vector<int4> tiles((size_t)ntiles);
    long long pi = 0, pk = 0;
    for (long long t = 1; t <= ntiles; ++t) {
        long long i, k;
        if (t == ntiles) { i = n; k = nnz; }
        else {
            const long long d = t * D;
            long long lo = std::max(0ll, d - nnz), hi = std::min(d, n);
            while (lo < hi) {
                const long long mid = (lo + hi) >> 1;
                if ((long long)rp[mid + 1] <= d - mid - 1) lo = mid + 1; else hi = mid;
            }
            i = lo; k = d - lo;
            const long long k4 = std::min(nnz, (k + 3) & ~3ll);
            if (k4 > k) {
                i = std::lower_bound(rp.begin() + i + 1, rp.begin() + n + 1, (int32_t)k4) - (rp.begin() + 1);
                k = k4;
            }
            if (i > n) i = n;
            if (i < pi || k < pk) { i = pi; k = pk; }
        }
        tiles[(size_t)t - 1] = make_int4((int)pi, (int)i, (int)pk, (int)k);
        pi = i; pk = k;
    }
    const size_t cb = 2 * (size_t)ntiles * elem_bytes(A->dtype);
    CU(cudaMalloc(&A->d_aux, sizeof(int4) * tiles.size()));
    CU(cudaMemcpy(A->d_aux, tiles.data(), sizeof(int4) * tiles.size(), cudaMemcpyHostToDevice));
    CU(cudaMalloc(&A->d_carry, cb));
    CU(cudaMemset(A->d_carry, 0, cb));
    A->dev.aux = (const int32_t*)A->d_aux;
    A->dev.aux_count = (int)ntiles;
    A->dev.carry = A->d_carry;
    A->kernel = KERNEL_MERGE;
    return MSOLVE_OK;
}

extern "C" int msolve_create_csr(msolve_matrix** out, int64_t n, int64_t nnz, const int32_t* d_rowptr,
                                 const int32_t* d_colidx, const void* d_val, int dtype, int flags, void* stream) {
    if (!out) return fail(MSOLVE_EINVAL, "msolve_create_csr: A is NULL");
    *out = nullptr;
    if (n < 0 || nnz < 0 || nnz >= (1ll << 31) || n >= (1ll << 31)) return fail(MSOLVE_EINVAL, "msolve_create_csr: bad n/nnz");
    if (!d_rowptr || (nnz > 0 && (!d_colidx || !d_val))) return fail(MSOLVE_EINVAL, "msolve_create_csr: NULL array");
    if (!valid_dtype(dtype)) return fail(MSOLVE_EINVAL, "msolve_create_csr: bad dtype");
    if (flags < MSOLVE_SPMV_AUTO || flags > MSOLVE_SPMV_TILE) return fail(MSOLVE_EINVAL, "msolve_create_csr: bad flags");
    if (!aligned16(d_val) || ((uintptr_t)d_colidx & 3u) || ((uintptr_t)d_rowptr & 3u)) return fail(MSOLVE_EINVAL, "msolve_create_csr: misaligned array");
    msolve_matrix* A = new (std::nothrow) msolve_matrix();
    if (!A) return fail(MSOLVE_ENOMEM, "out of host memory");
    A->format = FMT_CSR;
    A->dtype = dtype;
    A->dev.rowptr = d_rowptr; A->dev.colidx = d_colidx; A->dev.val = d_val;
    A->dev.n = n; A->dev.nbrows = 0; A->dev.nnz = nnz; A->dev.aux = nullptr; A->dev.aux_count = 0; A->dev.carry = nullptr;
    A->kernel = KERNEL_VECTOR;
    A->dev.x_pin = elem_bytes(dtype) <= 8 && (size_t)n * elem_bytes(dtype) <= (size_t)48 << 20;
    const double mean = n > 0 ? (double)nnz / (double)n : 0.0;
    A->lanes = mean > 48 ? 32 : mean > 20 ? 8 : mean > 6 ? 4 : 2;
    int rc = create_common(out, A, (cudaStream_t)stream);
    if (rc == MSOLVE_OK && flags != MSOLVE_SPMV_VECTOR && n > 0) {
        const bool force = flags != MSOLVE_SPMV_AUTO;
        if (!aligned16(d_rowptr) || !aligned16(d_colidx)) {
            if (force) rc = fail(MSOLVE_EINVAL, "msolve_create_csr: the TMA-staged kernels need 16-byte aligned rowptr / colidx");
        } else {
            std::vector<int32_t> rp((size_t)n + 1);
            cudaError_t e = cudaMemcpy(rp.data(), d_rowptr, sizeof(int32_t) * (size_t)(n + 1), cudaMemcpyDeviceToHost);
            if (e != cudaSuccess) rc = fail(MSOLVE_ECUDA, "msolve_create_csr: reading rowptr failed: %s", cudaGetErrorString(e));
            else rc = build_merge_tiles(A, flags, rp);
        }
    }
    if (rc != MSOLVE_OK) { msolve_destroy(A); *out = nullptr; }
    return rc;
}

extern "C" int msolve_create_bsr3(msolve_matrix** out, int64_t nbrows, int64_t nblocks, const int32_t* d_browptr,
                                  const int32_t* d_bcolidx, const void* d_blocks, int dtype, int flags, void* stream) {
    if (!out) return fail(MSOLVE_EINVAL, "msolve_create_bsr3: A is NULL");
    *out = nullptr;
    if (nbrows < 0 || nblocks < 0 || nblocks >= (1ll << 31) / 9 || 3 * nbrows >= (1ll << 31)) return fail(MSOLVE_EINVAL, "msolve_create_bsr3: bad sizes");
    if (!d_browptr || (nblocks > 0 && (!d_bcolidx || !d_blocks))) return fail(MSOLVE_EINVAL, "msolve_create_bsr3: NULL array");
    if (!complex_dtype(dtype)) return fail(MSOLVE_EINVAL, "msolve_create_bsr3: dtype must be MSOLVE_C64 or MSOLVE_C128 (SU(3) blocks are complex)");
    if (flags != MSOLVE_SPMV_AUTO && flags != MSOLVE_SPMV_VECTOR) return fail(MSOLVE_EINVAL, "msolve_create_bsr3: bad flags");
    if (!aligned16(d_blocks) || ((uintptr_t)d_bcolidx & 3u) || ((uintptr_t)d_browptr & 3u)) return fail(MSOLVE_EINVAL, "msolve_create_bsr3: misaligned array");
    msolve_matrix* A = new (std::nothrow) msolve_matrix();
    if (!A) return fail(MSOLVE_ENOMEM, "out of host memory");
    A->format = FMT_BSR3;
    A->dtype = dtype;
    A->dev.rowptr = d_browptr; A->dev.colidx = d_bcolidx; A->dev.val = d_blocks;
    A->dev.n = 3 * nbrows; A->dev.nbrows = nbrows; A->dev.nnz = nblocks; A->dev.aux = nullptr; A->dev.aux_count = 0; A->dev.carry = nullptr;
    A->kernel = KERNEL_BSR_ROWS;
    int rc = create_common(out, A, (cudaStream_t)stream);
    // the TMA-staged kernel bulk-copies the block-column indices: they must be 16-byte aligned too (a torch
    // slice may not be); otherwise the row kernel
    if (rc == MSOLVE_OK && flags == MSOLVE_SPMV_AUTO && nbrows > 0 && aligned16(d_bcolidx)) rc = build_bsr_tiles(A);
    if (rc != MSOLVE_OK) { msolve_destroy(A); *out = nullptr; }
    return rc;
}

extern "C" int msolve_create_lattice_su3(msolve_matrix** out, int ndim, const int32_t* h_extents, const void* d_links,
                                         double diag, double c_f, double c_b, int dtype, int flags, void* stream) {
    if (!out) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: A is NULL");
    *out = nullptr;
    if (ndim < 1 || ndim > 4 || !h_extents) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: ndim must be in [1, 4]");
    long long vol = 1;
    for (int mu = 0; mu < ndim; ++mu) {
        if (h_extents[mu] < 1) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: extents must be >= 1");
        vol *= h_extents[mu];
        if (3 * vol >= (1ll << 31)) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: lattice too large (3 V >= 2^31)");
    }
    if (!d_links) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: NULL array");
    if (!complex_dtype(dtype)) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: dtype must be MSOLVE_C64 or MSOLVE_C128");
    if (flags != MSOLVE_SPMV_AUTO && flags != MSOLVE_SPMV_VECTOR) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: bad flags");
    if (!aligned16(d_links)) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: misaligned array");
    if (!std::isfinite(diag) || !std::isfinite(c_f) || !std::isfinite(c_b)) return fail(MSOLVE_EINVAL, "msolve_create_lattice_su3: non-finite coefficient");
    msolve_matrix* A = new (std::nothrow) msolve_matrix();
    if (!A) return fail(MSOLVE_ENOMEM, "out of host memory");
    A->format = FMT_LATTICE;
    A->dtype = dtype;
    A->dev.rowptr = nullptr; A->dev.colidx = nullptr; A->dev.val = d_links;
    A->dev.n = 3 * vol; A->dev.nbrows = vol; A->dev.nnz = (long long)ndim * vol;
    A->dev.aux = nullptr; A->dev.aux_count = 0; A->dev.carry = nullptr;
    A->dev.lat_ndim = ndim;
    for (int mu = 0; mu < 4; ++mu) A->dev.lat_ext[mu] = mu < ndim ? h_extents[mu] : 1;
    A->dev.lat_vol = vol;
    A->dev.lat_diag = diag; A->dev.lat_cf = c_f; A->dev.lat_cb = c_b;
    A->dev.lat_rows_per_tile = 1;
    A->kernel = KERNEL_LAT_ROWS;
    // TMA tile kernel: every x0-row of links / x must be a 16-byte multiple and fit a tile
    const int L0 = h_extents[0];
    const int NS = dtype == MSOLVE_C128 ? LatTile<double2>::NS : LatTile<float2>::NS;
    const bool row16 = ((size_t)L0 * 3 * elem_bytes(dtype)) % 16 == 0;
    if (flags == MSOLVE_SPMV_AUTO && row16 && L0 <= NS) {
        const int T = NS / L0;
        const long long nrows = vol / L0;
        A->dev.lat_rows_per_tile = T;
        A->dev.aux_count = (int)((nrows + T - 1) / T);
        A->kernel = KERNEL_LAT_TMA;
    }
    int rc = create_common(out, A, (cudaStream_t)stream);
    if (rc != MSOLVE_OK) { msolve_destroy(A); *out = nullptr; }
    return rc;
}

extern "C" void msolve_destroy(msolve_matrix* A) {
    if (!A) return;
    for (int i = 0; i < 2; ++i) {
        if (A->graphs[i].exec) cudaGraphExecDestroy(A->graphs[i].exec);
        if (A->graphs[i].graph) cudaGraphDestroy(A->graphs[i].graph);
    }
    if (A->capture_stream) cudaStreamDestroy(A->capture_stream);
    if (A->d_state) cudaFree(A->d_state);
    if (A->h_stage) cudaFreeHost(A->h_stage);
    if (A->d_aux) cudaFree(A->d_aux);
    if (A->d_carry) cudaFree(A->d_carry);
    if (A->d_host_buf) cudaFree(A->d_host_buf);
    if (A->d_batch_buf) cudaFree(A->d_batch_buf);
    for (int i = 0; i < 2; ++i) {
        if (A->ev_solved[i]) cudaEventDestroy(A->ev_solved[i]);
        if (A->ev_copied[i]) cudaEventDestroy(A->ev_copied[i]);
        if (A->ev_loaded[i]) cudaEventDestroy(A->ev_loaded[i]);
    }
    if (A->copy_stream) cudaStreamDestroy(A->copy_stream);
    if (A->h2d_stream) cudaStreamDestroy(A->h2d_stream);
    delete A;
}

extern "C" const char* msolve_last_error(void) { return g_err; }

extern "C" int msolve_config(msolve_matrix* A, int key, int value) {
    if (!A) return fail(MSOLVE_EINVAL, "msolve_config: A is NULL");
    if (key == MSOLVE_CFG_LOOP_MODE && (value == 0 || value == 1)) { A->opt.loop_mode = value; return MSOLVE_OK; }
    if (key == MSOLVE_CFG_UPDATE_KERNEL && (value == 0 || value == 1)) { A->opt.update_kernel = value; return MSOLVE_OK; }
    if (key == MSOLVE_CFG_LATTICE_KERNEL && value >= 0 && value <= 4) { A->opt.lattice_kernel = value; return MSOLVE_OK; }
    if (key == MSOLVE_CFG_STOP_RULE && (value == 0 || value == 1)) { A->opt.stop_rule = value; return MSOLVE_OK; }
    if (key == MSOLVE_CFG_ITER_PATH && value >= 0 && value <= 3) { A->opt.iter_path = value; return MSOLVE_OK; }
    if (key == MSOLVE_CFG_FUSED_CTAS && value >= 0 && value <= kFusedMaxCtas) { A->opt.fused_ctas = value; return MSOLVE_OK; }
    if (key == MSOLVE_CFG_MATRIX_L2 && value >= 0 && value <= 2) {
        A->opt.matrix_l2 = value;
        A->dev.mat_keep = value == 2 ? 100 : 0;
        return MSOLVE_OK;
    }
    if (key == MSOLVE_CFG_DEFER_UPDATE && value >= 0 && value <= kDeferMax) { A->opt.defer = value; return MSOLVE_OK; }
    if (key == MSOLVE_CFG_MATRIX_L2_KEEP_PERCENT && value >= 0 && value <= 100) { A->dev.mat_keep = value; return MSOLVE_OK; }
    if (key == MSOLVE_CFG_X_WINDOW && (value == 0 || value == 1)) {
        if (value == 1) {
            if (A->format != FMT_CSR || A->kernel != KERNEL_VECTOR) return fail(MSOLVE_EINVAL, "msolve_config: MSOLVE_CFG_X_WINDOW applies to the vector-CSR kernel");
            int dev_max = 0, win_max = 0;
            CU(cudaDeviceGetAttribute(&dev_max, cudaDevAttrMaxPersistingL2CacheSize, A->device));
            CU(cudaDeviceGetAttribute(&win_max, cudaDevAttrMaxAccessPolicyWindowSize, A->device));
            if (dev_max <= 0 || win_max <= 0) return fail(MSOLVE_EINVAL, "msolve_config: the device has no persisting L2");
            const size_t want = std::min<size_t>((size_t)dev_max, (size_t)A->dev.n * elem_bytes(A->dtype));
            CU(cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want));     // device-wide set-aside
            A->l2_persist_bytes = want;
            A->l2_window_max = (size_t)win_max;
        }
        A->opt.x_window = value;
        return MSOLVE_OK;
    }
    return fail(MSOLVE_EINVAL, "msolve_config: bad key/value");
}

extern "C" int msolve_set_history(msolve_matrix* A, double* d_hist, int cap_rows) {
    if (!A) return fail(MSOLVE_EINVAL, "msolve_set_history: A is NULL");
    if (cap_rows < 0 || (cap_rows > 0 && !d_hist) || ((uintptr_t)d_hist & 7u)) return fail(MSOLVE_EINVAL, "msolve_set_history: bad buffer");
    A->d_hist = cap_rows > 0 ? d_hist : nullptr;
    A->hist_cap = cap_rows > 0 ? cap_rows : 0;
    return MSOLVE_OK;
}

extern "C" int msolve_set_phase_clock(msolve_matrix* A, uint64_t* d_ns) {
    if (!A) return fail(MSOLVE_EINVAL, "msolve_set_phase_clock: A is NULL");
    if ((uintptr_t)d_ns & 7u) return fail(MSOLVE_EINVAL, "msolve_set_phase_clock: d_ns must be 8-byte aligned");
    A->d_phase_ns = (unsigned long long*)d_ns;
    return MSOLVE_OK;
}

extern "C" int64_t msolve_last_launch_count(const msolve_matrix* A) { return A ? A->last_launches : 0; }

extern "C" const char* msolve_kernel_name(int alg, int j) {
    if (alg == MSOLVE_ALG_CGM && j >= 0 && j < 6) return kCgmNames[j];
    if (alg == MSOLVE_ALG_BICGSTABM && j >= 0 && j < 7) return kBiNames[j];
    return "";
}

// ------------------------------------------------------------------------------------- workspace
long long msolve::pk_stride_elems(const msolve_matrix* A) { return (long long)align_up((size_t)A->dev.n, 16); }
static int base_vectors(int alg) { return alg == MSOLVE_ALG_CGM ? 3 : 5; }  // r p q [s t]

extern "C" size_t msolve_workspace_bytes(const msolve_matrix* A, int nshifts, int algorithm) {
    if (!A || nshifts < 1 || nshifts > kMaxShifts || (algorithm != MSOLVE_ALG_CGM && algorithm != MSOLVE_ALG_BICGSTABM)) return 0;
    const size_t vb = align_up((size_t)pk_stride_elems(A) * elem_bytes(A->dtype), 256);
    // the deferred update keeps r in a ring of defer + 1 vectors (defer more than the one r of the step-by-step form)
    return vb * (size_t)(base_vectors(algorithm) + nshifts + defer_len(A, algorithm)) + 256;
}

static int fill_header(const msolve_matrix* A, int alg, const void* d_b, const double* h_shifts, int S, double tol,
                       int max_iter, void* d_x, void* ws, size_t ws_bytes, int force_all, SolveHeader* h) {
    if (!A) return fail(MSOLVE_EINVAL, "solve: A is NULL");
    if (S < 1 || S > kMaxShifts) return fail(MSOLVE_EINVAL, "solve: nshifts must be in [1, %d]", kMaxShifts);
    if (!d_b || !d_x || !h_shifts || !ws) return fail(MSOLVE_EINVAL, "solve: NULL argument");
    if (!(tol >= 0.0) || max_iter < 0) return fail(MSOLVE_EINVAL, "solve: bad tol / max_iter");
    if (!aligned16(d_b) || !aligned16(d_x)) return fail(MSOLVE_EINVAL, "solve: d_b / d_x must be 16-byte aligned");
    const size_t need = msolve_workspace_bytes(A, S, alg);
    if (ws_bytes < need) return fail(MSOLVE_ENOMEM, "solve: workspace too small (%zu < %zu)", ws_bytes, need);
    const size_t vb = align_up((size_t)pk_stride_elems(A) * elem_bytes(A->dtype), 256);
    char* base = (char*)align_up((size_t)(uintptr_t)ws, 256);
    memset(h, 0, sizeof(*h));
    h->b = d_b; h->x = d_x;
    const int defer = defer_len(A, alg);
    h->r = base; h->p = base + vb; h->q = base + 2 * vb;
    char* next = base + 3 * vb;
    if (alg == MSOLVE_ALG_BICGSTABM) { h->s = next; h->t = next + vb; next += 2 * vb; }
    h->pk = next;
    if (defer > 0) {                              // the ring of defer + 1 residuals: r's own vector and the defer extra ones
        h->p = base; h->q = base + vb; h->pk = base + 2 * vb;
        h->ring = base + (size_t)(2 + S) * vb;
        h->ring_stride = (long long)vb;
        h->r = h->ring;                           // r_0 = slot 0
    }
    h->n = A->dev.n;
    h->pk_stride = pk_stride_elems(A);
    h->x_stride = A->dev.n;
    h->tol = tol; h->S = S; h->max_iter = max_iter; h->force_all = force_all;
    h->defer = defer;
    h->stop_rule = A->opt.stop_rule; h->hist = A->d_hist; h->hist_cap = A->hist_cap; h->phase_ns = A->d_phase_ns;
    for (int k = 0; k < S; ++k) h->sigma[k] = h_shifts[k];
    return MSOLVE_OK;
}

static void fill_result_init(SolveResult* r, int S) {
    memset(r, 0, sizeof(*r));
    r->nactive = S;
    for (int k = 0; k < kMaxShifts; ++k) { r->conv_iter[k] = -1; r->relres[k] = 1.0; }
}

// ------------------------------------------------------------------------------------- solve
int msolve::run_solver(int alg, const msolve_matrix* Ac, const void* d_b, const double* h_shifts, int S, double tol,
                       int max_iter, void* d_x, void* ws, size_t ws_bytes, int* h_iterations, int* h_conv_iter,
                       double* h_relres, void* stream_, int per_shift_norm) {
    msolve_matrix* A = const_cast<msolve_matrix*>(Ac);
    if (!A) return fail(MSOLVE_EINVAL, "solve: A is NULL");
    int rc = check_device(A, "solve");
    if (rc != MSOLVE_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    SolveHeader* hh = &A->h_stage->h;
    SolveResult* hr = &A->h_stage->res;
    rc = fill_header(A, alg, d_b, h_shifts, S, tol, max_iter, d_x, ws, ws_bytes, 0, hh);
    if (rc != MSOLVE_OK) return rc;
    hh->per_shift_norm = per_shift_norm;
    fill_result_init(hr, S);
    const size_t xbytes = (size_t)S * (size_t)A->dev.n * elem_bytes(A->dtype);
    if (A->dev.n == 0 || max_iter == 0) {  // nothing to iterate: x = 0
        CU(cudaMemsetAsync(d_x, 0, xbytes, stream));
        CU(cudaStreamSynchronize(stream));
        if (h_iterations) *h_iterations = 0;
        for (int k = 0; k < S; ++k) { if (h_conv_iter) h_conv_iter[k] = A->dev.n == 0 ? 0 : -1; if (h_relres) h_relres[k] = A->dev.n == 0 ? 0.0 : 1.0; }
        A->last_launches = 0;
        return A->dev.n == 0 ? MSOLVE_OK : MSOLVE_MAXITER;
    }
    const int mode = A->opt.loop_mode;
    // Systems that live in L2 are bound by launch latency, not bytes: the whole solve runs as ONE cooperative
    // kernel (fused_small.cu).  AUTO: matrix + (4 + 2 S) vectors at most kFusedMaxBytes.
    // the smallest systems (a few MB) even fit in the shared memory of the 148 SMs: resident.cu (CG-M, CSR / BSR3)
    bool resident = false;
    if ((A->opt.iter_path == 3 || A->opt.iter_path == 0) && (A->format == FMT_CSR || A->format == FMT_BSR3) &&
        matrix_bytes(A) + (size_t)(3 + 2 * S) * (size_t)A->dev.n * elem_bytes(A->dtype) <= kResidentMaxBytes) {
        const size_t units = A->format == FMT_BSR3 ? (size_t)A->dev.nbrows : (size_t)A->dev.n;
        if (A->h_rowptr.size() != units + 1) {
            A->h_rowptr.resize(units + 1);
            CU(cudaMemcpyAsync(A->h_rowptr.data(), A->dev.rowptr, sizeof(int32_t) * (units + 1), cudaMemcpyDeviceToHost, stream));
            CU(cudaStreamSynchronize(stream));
        }
        resident = resident_supported(A, S, alg);
    }
    if (A->opt.iter_path == 3 && !resident) return fail(MSOLVE_EINVAL, "solve: MSOLVE_CFG_ITER_PATH = 3 needs a CSR / BSR3 handle whose matrix and vectors fit in shared memory");
    const bool fused = resident || A->opt.iter_path == 2 ||
                       (A->opt.iter_path == 0 && fused_supported(A) &&
                        matrix_bytes(A) + (size_t)(4 + 2 * S) * (size_t)A->dev.n * elem_bytes(A->dtype) <=
                            (defer_len(A, alg) > 0 ? kFusedMaxBytesDeferred : kFusedMaxBytes));
    if (fused) {
        if (!resident && !fused_supported(A)) return fail(MSOLVE_EINVAL, "solve: MSOLVE_CFG_ITER_PATH = 2 needs a vector-CSR, BSR3 or lattice handle, the register update kernel and the WHILE loop mode");
        // the header travels as a kernel argument and the kernel initialises the result block itself: no H2D copy
        rc = resident ? launch_resident(A, S, alg, stream) : launch_fused(A, alg, stream);
        if (rc != MSOLVE_OK) return rc;
        CU(cudaMemcpyAsync(hr, &A->d_state->res, sizeof(SolveResult), cudaMemcpyDeviceToHost, stream));
        CU(cudaStreamSynchronize(stream));
        if (hr->zero_rhs || (hr->status == MSOLVE_BREAKDOWN && hr->n_iter == 0)) {
            CU(cudaMemsetAsync(d_x, 0, xbytes, stream));
            CU(cudaStreamSynchronize(stream));
        }
        A->last_launches = 1;
        if (h_iterations) *h_iterations = hr->n_iter;
        for (int k = 0; k < S; ++k) {
            if (h_conv_iter) h_conv_iter[k] = hr->conv_iter[k];
            if (h_relres) h_relres[k] = hr->relres[k];
        }
        return hr->status;
    }
    rc = build_graph(A, alg);
    if (rc != MSOLVE_OK) return rc;
    CU(cudaMemcpyAsync(A->d_state, A->h_stage, sizeof(SolveHeader) + sizeof(SolveResult), cudaMemcpyHostToDevice, stream));
    rc = launch_init(A, stream);
    if (rc != MSOLVE_OK) return rc;
    CU(cudaGetLastError());
    int64_t launches = 2;
    if (mode == 0) {
        CU(cudaGraphLaunch(A->graphs[alg].exec, stream));
        CU(cudaMemcpyAsync(hr, &A->d_state->res, sizeof(SolveResult), cudaMemcpyDeviceToHost, stream));
        CU(cudaStreamSynchronize(stream));
        launches += (int64_t)launches_per_iter(A, alg) * std::max(1, hr->n_iter + (hr->status == MSOLVE_BREAKDOWN ? 1 : 0));
    } else {
        for (;;) {
            CU(cudaGraphLaunch(A->graphs[alg].exec, stream));
            launches += (int64_t)launches_per_iter(A, alg) * kChunk;
            CU(cudaMemcpyAsync(hr, &A->d_state->res, sizeof(SolveResult), cudaMemcpyDeviceToHost, stream));
            CU(cudaStreamSynchronize(stream));
            if (hr->done) break;
        }
    }
    // x_k = 0 is substituted in registers until the first update has written it: b = 0 and a breakdown in the
    // first loop body (before any update) leave d_x untouched, so it is zeroed here (the iterate IS x_k = 0)
    if (hr->zero_rhs || (hr->status == MSOLVE_BREAKDOWN && hr->n_iter == 0)) {
        CU(cudaMemsetAsync(d_x, 0, xbytes, stream));
        CU(cudaStreamSynchronize(stream));
    }
    A->last_launches = launches;
    if (h_iterations) *h_iterations = hr->n_iter;
    for (int k = 0; k < S; ++k) {
        if (h_conv_iter) h_conv_iter[k] = hr->conv_iter[k];
        if (h_relres) h_relres[k] = hr->relres[k];
    }
    return hr->status;
}

extern "C" int msolve_cgm(const msolve_matrix* A, const void* d_b, const double* h_shifts, int nshifts, double tol,
                          int max_iter, void* d_x, void* d_workspace, size_t workspace_bytes, int* h_iterations,
                          int* h_conv_iter, double* h_relres, void* stream) {
    return run_solver(MSOLVE_ALG_CGM, A, d_b, h_shifts, nshifts, tol, max_iter, d_x, d_workspace, workspace_bytes,
                      h_iterations, h_conv_iter, h_relres, stream, 0);
}

extern "C" int msolve_bicgstabm(const msolve_matrix* A, const void* d_b, const double* h_shifts, int nshifts, double tol,
                                int max_iter, void* d_x, void* d_workspace, size_t workspace_bytes, int* h_iterations,
                                int* h_conv_iter, double* h_relres, void* stream) {
    return run_solver(MSOLVE_ALG_BICGSTABM, A, d_b, h_shifts, nshifts, tol, max_iter, d_x, d_workspace, workspace_bytes,
                      h_iterations, h_conv_iter, h_relres, stream, 0);
}

extern "C" int msolve_solve_host(const msolve_matrix* A, int algorithm, const void* h_b, const double* h_shifts,
                                 int nshifts, double tol, int max_iter, void* h_x, int* h_iterations,
                                 int* h_conv_iter, double* h_relres, void* stream_) {
    if (!A || !h_b || !h_x) return fail(MSOLVE_EINVAL, "msolve_solve_host: NULL argument");
    if (algorithm != MSOLVE_ALG_CGM && algorithm != MSOLVE_ALG_BICGSTABM) return fail(MSOLVE_EINVAL, "msolve_solve_host: bad algorithm");
    const size_t wsb = msolve_workspace_bytes(A, nshifts, algorithm);
    if (!wsb) return fail(MSOLVE_EINVAL, "msolve_solve_host: bad nshifts");
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t eb = elem_bytes(A->dtype);
    const size_t bbytes = (size_t)A->dev.n * eb, xbytes = bbytes * (size_t)nshifts;
    msolve_matrix* Am = const_cast<msolve_matrix*>(A);
    const size_t boff = 0, xoff = align_up(bbytes, 256), woff = xoff + align_up(xbytes, 256);
    if (Am->host_buf_bytes < woff + wsb + 256) {               // grow-only cache of the device buffers
        if (Am->d_host_buf) cudaFree(Am->d_host_buf);
        Am->d_host_buf = nullptr; Am->host_buf_bytes = 0;
        if (cudaMalloc((void**)&Am->d_host_buf, woff + wsb + 256) != cudaSuccess) return fail(MSOLVE_ENOMEM, "msolve_solve_host: cudaMalloc of %zu bytes failed", woff + wsb);
        Am->host_buf_bytes = woff + wsb + 256;
    }
    char* d_all = Am->d_host_buf;
    int rc;
    cudaError_t e = cudaMemcpyAsync(d_all + boff, h_b, bbytes, cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) return fail(MSOLVE_ECUDA, "H2D copy failed: %s", cudaGetErrorString(e));
    rc = run_solver(algorithm, A, d_all + boff, h_shifts, nshifts, tol, max_iter, d_all + xoff, d_all + woff, wsb + 256,
                    h_iterations, h_conv_iter, h_relres, stream_, 0);
    if (rc >= 0) {
        e = cudaMemcpyAsync(h_x, d_all + xoff, xbytes, cudaMemcpyDeviceToHost, stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) rc = fail(MSOLVE_ECUDA, "D2H copy failed: %s", cudaGetErrorString(e));
    }
    return rc;
}

// A batch of right-hand sides through the host interface, software-pipelined: the D2H copy of
// solve i (on a copy stream, out of x slot i % 2) overlaps solve i+1 (which writes the other slot).
extern "C" int msolve_solve_host_batch(const msolve_matrix* A, int algorithm, int nrhs, const void* const* h_b,
                                       const double* h_shifts, int nshifts, double tol, int max_iter,
                                       void* const* h_x, int* h_iterations, int* h_conv_iter, double* h_relres,
                                       void* stream_) {
    if (!A || !h_b || !h_x || nrhs < 0) return fail(MSOLVE_EINVAL, "msolve_solve_host_batch: bad argument");
    if (algorithm != MSOLVE_ALG_CGM && algorithm != MSOLVE_ALG_BICGSTABM) return fail(MSOLVE_EINVAL, "msolve_solve_host_batch: bad algorithm");
    for (int i = 0; i < nrhs; ++i)
        if (!h_b[i] || !h_x[i]) return fail(MSOLVE_EINVAL, "msolve_solve_host_batch: NULL vector %d", i);
    const size_t wsb = msolve_workspace_bytes(A, nshifts, algorithm);
    if (!wsb) return fail(MSOLVE_EINVAL, "msolve_solve_host_batch: bad nshifts");
    if (nrhs == 0) return MSOLVE_OK;
    cudaStream_t stream = (cudaStream_t)stream_;
    msolve_matrix* Am = const_cast<msolve_matrix*>(A);
    const size_t eb = elem_bytes(A->dtype);
    const size_t bbytes = (size_t)A->dev.n * eb, xbytes = bbytes * (size_t)nshifts;
    const size_t slot = align_up(bbytes, 256) + align_up(xbytes, 256);
    const size_t need = 2 * slot + wsb + 256;
    if (Am->batch_buf_bytes < need) {
        if (Am->d_batch_buf) cudaFree(Am->d_batch_buf);
        Am->d_batch_buf = nullptr; Am->batch_buf_bytes = 0;
        if (cudaMalloc((void**)&Am->d_batch_buf, need) != cudaSuccess) return fail(MSOLVE_ENOMEM, "msolve_solve_host_batch: cudaMalloc of %zu bytes failed", need);
        Am->batch_buf_bytes = need;
    }
    if (!Am->copy_stream) {
        CU(cudaStreamCreateWithFlags(&Am->copy_stream, cudaStreamNonBlocking));
        for (int j = 0; j < 2; ++j) {
            CU(cudaEventCreateWithFlags(&Am->ev_solved[j], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&Am->ev_copied[j], cudaEventDisableTiming));
        }
    }
    if (!Am->h2d_stream) {
        CU(cudaStreamCreateWithFlags(&Am->h2d_stream, cudaStreamNonBlocking));
        for (int j = 0; j < 2; ++j) CU(cudaEventCreateWithFlags(&Am->ev_loaded[j], cudaEventDisableTiming));
    }
    char* d_ws = Am->d_batch_buf + 2 * slot;
    int worst = MSOLVE_OK;
    // b_0 goes up front; b_{i+1} is sent on its own stream (the host-to-device copy engine) while solve i runs: the
    // b of slot (i+1) & 1 was last read by solve i-1, which has completed (run_solver synchronises `stream`)
    CU(cudaMemcpyAsync(Am->d_batch_buf, h_b[0], bbytes, cudaMemcpyHostToDevice, Am->h2d_stream));
    CU(cudaEventRecord(Am->ev_loaded[0], Am->h2d_stream));
    for (int i = 0; i < nrhs; ++i) {
        const int j = i & 1;
        char* d_b = Am->d_batch_buf + (size_t)j * slot;
        char* d_x = d_b + align_up(bbytes, 256);
        if (i + 1 < nrhs) {
            CU(cudaMemcpyAsync(Am->d_batch_buf + (size_t)(j ^ 1) * slot, h_b[i + 1], bbytes, cudaMemcpyHostToDevice, Am->h2d_stream));
            CU(cudaEventRecord(Am->ev_loaded[j ^ 1], Am->h2d_stream));
        }
        if (i >= 2) CU(cudaStreamWaitEvent(stream, Am->ev_copied[j], 0));       // slot j has been read back
        CU(cudaStreamWaitEvent(stream, Am->ev_loaded[j], 0));                    // b_i has arrived
        const int rc = run_solver(algorithm, A, d_b, h_shifts, nshifts, tol, max_iter, d_x, d_ws, wsb + 256,
                                  h_iterations ? h_iterations + i : nullptr,
                                  h_conv_iter ? h_conv_iter + (size_t)i * nshifts : nullptr,
                                  h_relres ? h_relres + (size_t)i * nshifts : nullptr, stream_, 0);
        if (rc < 0) { cudaStreamSynchronize(Am->copy_stream); cudaStreamSynchronize(Am->h2d_stream); return rc; }
        worst = std::max(worst, rc);
        CU(cudaEventRecord(Am->ev_solved[j], stream));
        CU(cudaStreamWaitEvent(Am->copy_stream, Am->ev_solved[j], 0));
        CU(cudaMemcpyAsync(h_x[i], d_x, xbytes, cudaMemcpyDeviceToHost, Am->copy_stream));
        CU(cudaEventRecord(Am->ev_copied[j], Am->copy_stream));
    }
    CU(cudaStreamSynchronize(Am->copy_stream));
    return worst;
}

// ------------------------------------------------------------------------------------- spmv / profile
extern "C" int msolve_spmv(const msolve_matrix* Ac, const void* d_x, void* d_y, double* h_dot, void* stream_) {
    msolve_matrix* A = const_cast<msolve_matrix*>(Ac);
    if (!A || !d_x || !d_y) return fail(MSOLVE_EINVAL, "msolve_spmv: NULL argument");
    if (!aligned16(d_x) || !aligned16(d_y)) return fail(MSOLVE_EINVAL, "msolve_spmv: d_x / d_y must be 16-byte aligned");
    int rc = check_device(A, "msolve_spmv");
    if (rc != MSOLVE_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    SolveHeader* hh = &A->h_stage->h;
    memset(hh, 0, sizeof(*hh));
    hh->sp_x = d_x; hh->sp_y = d_y; hh->sp_u = d_x; hh->n = A->dev.n; hh->S = 1;
    fill_result_init(&A->h_stage->res, 1);
    CU(cudaMemcpyAsync(A->d_state, A->h_stage, sizeof(SolveHeader) + sizeof(SolveResult), cudaMemcpyHostToDevice, stream));
    if (A->dev.n > 0 && (rc = launch_spmv<ROLE_GEN>(A, stream)) != MSOLVE_OK) return rc;
    CU(cudaGetLastError());
    if (h_dot) {
        h_dot[0] = h_dot[1] = 0.0;
        if (A->dev.n > 0) {
            int count = 0;
            CU(cudaMemcpyAsync(&count, &A->d_state->partial_count, sizeof(int), cudaMemcpyDeviceToHost, stream));
            CU(cudaStreamSynchronize(stream));
            double* tmp = new double[2 * kMaxPartials];
            cudaError_t e = cudaMemcpy(tmp, A->d_state->partial, sizeof(double) * 2 * kMaxPartials, cudaMemcpyDeviceToHost);
            if (e == cudaSuccess)
                for (int i = 0; i < count; ++i) { h_dot[0] += tmp[i]; h_dot[1] += tmp[kMaxPartials + i]; }
            delete[] tmp;
            if (e != cudaSuccess) return fail(MSOLVE_ECUDA, "msolve_spmv: D2H failed: %s", cudaGetErrorString(e));
        }
    } else {
        CU(cudaStreamSynchronize(stream));
    }
    return MSOLVE_OK;
}

extern "C" int msolve_profile_iteration(const msolve_matrix* Ac, int alg, const void* d_b, const double* h_shifts,
                                        int S, int iters, void* d_x, void* ws, size_t ws_bytes, float* h_ms,
                                        int* h_launches, void* stream_) {
    msolve_matrix* A = const_cast<msolve_matrix*>(Ac);
    if (!A) return fail(MSOLVE_EINVAL, "profile: A is NULL");
    if (alg != MSOLVE_ALG_CGM && alg != MSOLVE_ALG_BICGSTABM) return fail(MSOLVE_EINVAL, "profile: bad algorithm");
    if (iters < 1 || !h_ms) return fail(MSOLVE_EINVAL, "profile: bad iters / h_ms");
    cudaStream_t stream = (cudaStream_t)stream_;
    int rc = check_device(A, "profile");
    if (rc != MSOLVE_OK) return rc;
    rc = fill_header(A, alg, d_b, h_shifts, S, 0.0, iters + 1, d_x, ws, ws_bytes, 1, &A->h_stage->h);
    if (rc != MSOLVE_OK) return rc;
    fill_result_init(&A->h_stage->res, S);
    CU(cudaMemcpyAsync(A->d_state, A->h_stage, sizeof(SolveHeader) + sizeof(SolveResult), cudaMemcpyHostToDevice, stream));
    if ((rc = launch_init(A, stream)) != MSOLVE_OK) return rc;
    const int nk = kernels_per_iter(A, alg);
    cudaEvent_t ev[9];
    for (int j = 0; j <= nk; ++j) CU(cudaEventCreate(&ev[j]));
    double sum[8] = {0};
    // one untimed warm-up iteration (also leaves n_iter > 0 so the steady-state paths are timed)
    for (int it = 0; it <= iters; ++it) {
        for (int j = 0; j < nk; ++j) {
            CU(cudaEventRecord(ev[j], stream));
            if ((rc = launch_body_kernel(A, alg, j, stream, 0, 0)) != MSOLVE_OK) return rc;
        }
        CU(cudaEventRecord(ev[nk], stream));
        CU(cudaStreamSynchronize(stream));
        CU(cudaGetLastError());
        if (it == 0) continue;
        for (int j = 0; j < nk; ++j) {
            float ms = 0.f;
            CU(cudaEventElapsedTime(&ms, ev[j], ev[j + 1]));
            sum[j] += ms;
        }
    }
    for (int j = 0; j <= nk; ++j) cudaEventDestroy(ev[j]);
    for (int j = 0; j < 8; ++j) { h_ms[j] = j < nk ? (float)(sum[j] / iters) : 0.f; if (h_launches) h_launches[j] = j < nk ? 1 : 0; }
    if (h_launches && A->kernel == KERNEL_MERGE) {   // merge-path SpMV slots are two launches each
        if (alg == MSOLVE_ALG_CGM) h_launches[1] = 2; else { h_launches[0] = 2; h_launches[3] = 2; }
    }
    return nk;
}
