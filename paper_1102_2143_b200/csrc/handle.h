// handle.h -- host-side handle of the C ABI (include/msolve.h) and the launch interface between the
// translation units of libmsolve.so:
//   msolve.cu      C ABI, create/destroy, graph capture, solver drivers
//   spmv_role.cu   SpMV launches, compiled once per ROLE (the fused reductions differ per role)
//   vec.cu         vector-update and scalar-recurrence kernels
//   fused_small.cu whole solve as one cooperative kernel for systems that live in L2
//   resident.cu    whole solve with matrix and vectors resident in shared memory (systems of a few MB)
//   multirhs.cu    a right-hand side per shift, eq. (6)
//   slab.cu        row-partitioned operator (halo exchange between slabs)
#pragma once

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <vector>

#include "common.cuh"

namespace msolve {

enum { FMT_CSR = 0, FMT_BSR3 = 1, FMT_LATTICE = 2 };
enum { KERNEL_VECTOR = 1, KERNEL_MERGE = 2, KERNEL_BSR_ROWS = 3, KERNEL_BSR_TMA = 4, KERNEL_LAT_ROWS = 5, KERNEL_LAT_TMA = 6, KERNEL_CSR_TILE = 7 };
constexpr int kChunk = 8;  // iteration bodies per graph launch in chunked loop mode

// per-handle options (msolve_config)
struct Options {
    int loop_mode = 0;       // MSOLVE_CFG_LOOP_MODE
    int update_kernel = 0;   // MSOLVE_CFG_UPDATE_KERNEL
    int lattice_kernel = 0;  // MSOLVE_CFG_LATTICE_KERNEL
    int stop_rule = 0;       // MSOLVE_CFG_STOP_RULE
    int iter_path = 0;       // MSOLVE_CFG_ITER_PATH
    int x_window = 0;        // MSOLVE_CFG_X_WINDOW
    int matrix_l2 = 0;       // MSOLVE_CFG_MATRIX_L2
    int fused_ctas = 0;      // MSOLVE_CFG_FUSED_CTAS
    int defer = kDeferMax;   // MSOLVE_CFG_DEFER_UPDATE: chunk length of the deferred multishift update (0 = off)
    int graph_key() const { return loop_mode | (update_kernel << 1) | (lattice_kernel << 2) | (iter_path << 5) | (x_window << 7) | (defer << 8); }
};

struct LoopGraph {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    int key = -1;
    const void* xptr = nullptr;   // x_window: the vector the captured access-policy windows cover
    const void* xptr2 = nullptr;
};

}  // namespace msolve

struct msolve_slab_set;   // slab.cu

struct msolve_matrix {
    int format = msolve::FMT_CSR;
    int dtype = MSOLVE_C128;
    int kernel = msolve::KERNEL_VECTOR;
    int lanes = 8;
    int tile_u = 4;                     // KERNEL_CSR_TILE: non-zeros per lane
    msolve::MatDev dev{};
    int device = 0;
    int num_sms = 148;
    msolve::Options opt;
    msolve::SolveState* d_state = nullptr;      // library-owned
    msolve::SolveState* h_stage = nullptr;      // pinned staging for header / result
    void* d_aux = nullptr;              // library-owned auxiliary matrix data
    void* d_carry = nullptr;            // merge-path carries (library-owned)
    double* d_hist = nullptr;           // msolve_set_history: caller's device buffer (borrowed)
    int hist_cap = 0;
    unsigned long long* d_phase_ns = nullptr;   // msolve_set_phase_clock (borrowed)
    char* d_host_buf = nullptr;         // msolve_solve_host: device b, x and workspace, kept for the next call
    size_t host_buf_bytes = 0;
    char* d_batch_buf = nullptr;        // msolve_solve_host_batch: two (b, x) slots + workspace
    size_t batch_buf_bytes = 0;
    cudaStream_t copy_stream = nullptr; // D2H of solve i overlaps solve i+1
    cudaStream_t h2d_stream = nullptr;  // H2D of b_{i+1} overlaps solve i (the other copy engine)
    cudaEvent_t ev_solved[2] = {nullptr, nullptr}, ev_copied[2] = {nullptr, nullptr}, ev_loaded[2] = {nullptr, nullptr};
    cudaStream_t capture_stream = nullptr;
    msolve::LoopGraph graphs[2];
    int64_t last_launches = 0;
    long long x_stride = 0;             // slab handles: elements between x_k and x_{k+1} in the caller's array (0 = n)
    size_t l2_persist_bytes = 0;        // MSOLVE_CFG_X_WINDOW: persisting L2 set-aside / largest window of the device
    size_t l2_window_max = 0;
    mutable int flush_ctas_per_sm = 0;       // resident CTAs per SM of k_cgm_flush (0: not asked yet), vec.cu
    mutable std::vector<int32_t> h_rowptr;   // host copy of rowptr / browptr (resident.cu sizes its ranges from it), filled on demand
    mutable std::vector<const void*> smem_attr_done;   // kernels whose dynamic shared-memory limit is raised on `device`
    msolve_slab_set* slabs = nullptr;   // row-partitioned form (msolve_create_*_slabs)
};

namespace msolve {

int fail(int code, const char* fmt, ...);

#define MSOLVE_CU(call)                                                                                \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess)                                                                         \
            return ::msolve::fail(MSOLVE_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

// chunk length of the deferred multishift update this handle uses for `alg` (0: the update of every iteration):
// CG-M with the register update kernel; BiCGStab-M and the TMA-staged update kernel keep the step-by-step form
inline int defer_len(const msolve_matrix* A, int alg) {
    return (alg == MSOLVE_ALG_CGM && A->opt.update_kernel == 0) ? A->opt.defer : 0;
}

inline size_t elem_bytes(int dtype) { return dtype == MSOLVE_C128 ? 16 : dtype == MSOLVE_F32 ? 4 : 8; }

// Raise the dynamic shared-memory limit of `kernel` once per handle (the attribute belongs to the
// device the handle lives on; a handle is bound to one device).  MSOLVE_OK or MSOLVE_ECUDA.
int ensure_smem(const msolve_matrix* A, const void* kernel, int bytes);

template <typename K>
inline int blocks_per_sm(K kernel, int threads) {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, threads, 0) != cudaSuccess || nb < 1) nb = 1;
    return nb;
}
// persistent grid: enough CTAs for `work_items` at `items_per_cta`, capped at full occupancy
template <typename K>
inline int grid_for(const msolve_matrix* A, K kernel, long long work_items, long long items_per_cta) {
    const long long full = (long long)A->num_sms * blocks_per_sm(kernel, kThreads);
    const long long need = (work_items + items_per_cta - 1) / items_per_cta;
    long long g = need < full ? need : full;
    if (g < 1) g = 1;
    return (int)(g < kMaxPartials ? g : kMaxPartials);
}

// y = A x with the fused reductions of ROLE, on the vectors named in the handle's SolveState.
// Defined in spmv_role.cu (one translation unit per ROLE).  Returns MSOLVE_OK or an error code.
template <int ROLE> int launch_spmv(const msolve_matrix* A, cudaStream_t s);
// launches per SpMV (merge-path: tile kernel + carry fix-up)
inline int spmv_launches(const msolve_matrix* A) { return A->kernel == KERNEL_MERGE ? 2 : 1; }

// vec.cu: the non-SpMV kernels of the iteration body, by position j (msolve_kernel_name), and the two init kernels
int launch_vec_kernel(const msolve_matrix* A, int alg, int j, cudaStream_t s, cudaGraphConditionalHandle cond, int use_cond);
int launch_init(const msolve_matrix* A, cudaStream_t s);             // both init kernels
int launch_init_vectors(const msolve_matrix* A, cudaStream_t s);     // r <- b, p <- b, partial <b,b>
int launch_init_state(const msolve_matrix* A, cudaStream_t s);       // scalars from the summed partials

// fused_small.cu: the whole solve as ONE cooperative kernel (systems that live in L2)
bool fused_supported(const msolve_matrix* A);
int launch_fused(const msolve_matrix* A, int alg, cudaStream_t s);

// resident.cu: CG-M with matrix and vectors resident in shared memory (systems of a few MB)
bool resident_supported(const msolve_matrix* A, int S, int alg);
int launch_resident(const msolve_matrix* A, int S, int alg, cudaStream_t s);

// msolve.cu: pieces the other entry points (multirhs.cu, slab.cu) build on
long long pk_stride_elems(const msolve_matrix* A);
int check_device(const msolve_matrix* A, const char* who);
// per_shift_norm = 1: shift k stops at |zeta_k| ||r|| <= tol * rhs_norm[k] (device array, eq. (6)) instead of tol ||b||
int run_solver(int alg, const msolve_matrix* A, const void* d_b, const double* h_shifts, int S, double tol, int max_iter,
               void* d_x, void* ws, size_t ws_bytes, int* h_iterations, int* h_conv_iter, double* h_relres, void* stream,
               int per_shift_norm);

}  // namespace msolve
