// multirhs.cu -- a different right-hand side per shift, eq. (6), PAPER.md:228-232:
//
//        (A + sigma_i I) x_i = b_i ,   i = 0 .. S-1 .
//
// The paper states the idea ("a judicious choice of initial guesses can deliver the same initial residual for
// each of the linear systems ... involves a number of SpMV operations, and so it seems worthwhile to develop a
// routine capable of producing these initial guesses using the GPU, after which our solver could finish the
// solution") and cites [18], which is not available; DESIGN.md "Per-shift right-hand sides" derives the
// construction, S - 1 SpMVs:
//   d_m   = divided differences of the b_i over the shifts (Newton form of the vector polynomial G(s), G(sigma_i) = b_i)
//   u_{S-2} = d_{S-1};  u_{m-1} = d_m - (A + sigma_m) u_m (m = S-2 .. 1);  r0 = d_0 - (A + sigma_0) u_0
//   y_i   = sum_{m <= i} w_m(sigma_i) u_m,  w_m(s) = prod_{j<m} (s - sigma_j)     =>  b_i - (A + sigma_i) y_i = r0 for all i
//   one multishift solve (A + sigma_i) z_i = r0 from z_i = 0 (the unchanged CG-M / BiCGStab-M iteration), x_i = y_i + z_i.
// Everything runs on the device, in stream order, without a host synchronisation before the solver's own.
#include "handle.h"
#include "tuning.h"

namespace msolve {

// per-shift partial sums of ||b_k||^2: grid (kNormBlocks, S)
constexpr int kNormBlocks = 32;

template <typename E>
__global__ void __launch_bounds__(kThreads) k_mr_norm_partials(SolveState* st, const E* B, long long n) {
    const E* b = B + (long long)blockIdx.y * n;
    double acc[1] = {0.0};
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        acc[0] += cnorm2(b[i]);
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) st->partial[blockIdx.y * kNormBlocks + blockIdx.x] = acc[0];
}

// ||b_k|| (fixed-order sums) and the Newton weights w_m(sigma_i) = prod_{j<m} (sigma_i - sigma_j), row i of wtab
__global__ void __launch_bounds__(kThreads) k_mr_norms_weights(SolveState* st, double* wtab, int S) {
    for (int k = threadIdx.x; k < S; k += blockDim.x) {
        double s = 0.0;
        for (int j = 0; j < kNormBlocks; ++j) s += st->partial[k * kNormBlocks + j];
        st->rhs_norm[k] = sqrt(s);
        double w = 1.0;
        for (int m = 0; m < S; ++m) { wtab[(size_t)k * S + m] = w; w *= st->h.sigma[k] - st->h.sigma[m]; }
    }
}

// D <- B, then the divided-difference table per element, in place: after level l, D[i] = b[sigma_{i-l} .. sigma_i].
// NMAX = 16: the column lives in registers (fully unrolled); NMAX = kMaxShifts: local memory.
template <typename E, int NMAX>
__global__ void __launch_bounds__(kThreads) k_mr_divdiff(SolveState* st, const E* B, E* D, long long n, long long stride, int S) {
    typedef typename RealOf<E>::type T;
    __shared__ double sg[kMaxShifts];
    for (int k = threadIdx.x; k < S; k += blockDim.x) sg[k] = st->h.sigma[k];
    __syncthreads();
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        E v[NMAX];
#pragma unroll
        for (int i = 0; i < NMAX; ++i) if (i < S) v[i] = B[(long long)i * n + e];
#pragma unroll
        for (int l = 1; l < NMAX; ++l) {
            if (l >= S) break;
#pragma unroll
            for (int i = NMAX - 1; i >= 1; --i) {
                if (i < l || i >= S) continue;
                const T inv = (T)(1.0 / (sg[i] - sg[i - l]));
                E d = csub(v[i], v[i - 1]);
                v[i] = clin_r(inv, d, (T)0, d);
            }
        }
#pragma unroll
        for (int i = 0; i < NMAX; ++i) if (i < S) D[(long long)i * stride + e] = v[i];
    }
}

// same table, any S, one level per pass over global memory (used when S > 16: the column does not fit registers)
template <typename E>
__global__ void __launch_bounds__(kThreads) k_mr_divdiff_level(SolveState* st, E* D, long long n, long long stride, int S, int l) {
    typedef typename RealOf<E>::type T;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        E hi = D[(long long)(S - 1) * stride + e];
        for (int i = S - 1; i >= l; --i) {
            const E lo = D[(long long)(i - 1) * stride + e];
            const T inv = (T)(1.0 / (st->h.sigma[i] - st->h.sigma[i - l]));
            const E d = csub(hi, lo);
            D[(long long)i * stride + e] = clin_r(inv, d, (T)0, d);
            hi = lo;
        }
    }
}

template <typename E>
__global__ void __launch_bounds__(kThreads) k_mr_copy(const E* B, E* D, long long n, long long stride, int S) {
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x)
        for (int i = 0; i < S; ++i) D[(long long)i * stride + e] = B[(long long)i * n + e];
}

// point the generic SpMV role at (x, y) in stream order
__global__ void k_mr_set_spmv(SolveState* st, const void* x, void* y) { st->h.sp_x = x; st->h.sp_y = y; st->h.sp_u = x; }

// dst <- dst - (q + sigma_m u)          (u_{m-1} = d_m - (A + sigma_m) u_m with q = A u_m)
template <typename E>
__global__ void __launch_bounds__(kThreads) k_mr_usub(SolveState* st, E* dst, const E* q, const E* u, long long n, int m) {
    typedef typename RealOf<E>::type T;
    const T sg = (T)st->h.sigma[m];
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x)
        dst[e] = csub(dst[e], caxpy_r(q[e], sg, u[e]));
}

// x_i <- x_i + sum_{m <= min(i, S-2)} w_m(sigma_i) u_m, m ascending (the order of the oracle).  S <= 16: the u_m of
// an element are read once into registers.
template <typename E>
__global__ void __launch_bounds__(kThreads) k_mr_add_guess16(E* x, const E* U, const double* wtab, long long n, long long stride, int S) {
    typedef typename RealOf<E>::type T;
    constexpr int NMAX = 16;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        E u[NMAX];
#pragma unroll
        for (int m = 0; m < NMAX; ++m) if (m < S - 1) u[m] = U[(long long)m * stride + e];
#pragma unroll
        for (int i = 0; i < NMAX; ++i) {
            if (i >= S) break;
            E xi = x[(long long)i * n + e];
#pragma unroll
            for (int m = 0; m < NMAX; ++m) {
                if (m > i || m > S - 2) break;
                xi = caxpy_r(xi, (T)wtab[(size_t)i * S + m], u[m]);
            }
            x[(long long)i * n + e] = xi;
        }
    }
}
// any S: u_m re-read through L1/L2
template <typename E>
__global__ void __launch_bounds__(kThreads) k_mr_add_guess(E* x, const E* U, const double* wtab, long long n, long long stride, int S) {
    typedef typename RealOf<E>::type T;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x)
        for (int i = 0; i < S; ++i) {
            E xi = x[(long long)i * n + e];
            for (int m = 0; m <= i && m <= S - 2; ++m) xi = caxpy_r(xi, (T)wtab[(size_t)i * S + m], U[(long long)m * stride + e]);
            x[(long long)i * n + e] = xi;
        }
}

// the shifts, passed by value, into the device-resident header (the setup kernels run before the solver stages its own)
struct SigmaArg { double v[kMaxShifts]; };
__global__ void k_mr_set_sigma(SolveState* st, SigmaArg sg, int S) {
    for (int k = threadIdx.x; k < S; k += blockDim.x) st->h.sigma[k] = sg.v[k];
    if (threadIdx.x == 0) st->h.S = S;
}

template <typename E>
static int multirhs_setup(const msolve_matrix* A, const void* d_B, int S, char* d_slots, long long stride, double* d_wtab, void* d_q, cudaStream_t s) {
    SolveState* st = A->d_state;
    const long long n = A->dev.n;
    const E* B = (const E*)d_B;
    E* D = (E*)d_slots;
    const int grid = (int)std::max(1ll, std::min<long long>((long long)A->num_sms * 4, (n + kThreads - 1) / kThreads));
    k_mr_norm_partials<E><<<dim3(kNormBlocks, S), kThreads, 0, s>>>(st, B, n);
    k_mr_norms_weights<<<1, kThreads, 0, s>>>(st, d_wtab, S);
    if (S <= 16) k_mr_divdiff<E, 16><<<grid, kThreads, 0, s>>>(st, B, D, n, stride, S);
    else {
        k_mr_copy<E><<<grid, kThreads, 0, s>>>(B, D, n, stride, S);
        for (int l = 1; l < S; ++l) k_mr_divdiff_level<E><<<grid, kThreads, 0, s>>>(st, D, n, stride, S, l);
    }
    for (int m = S - 2; m >= 0; --m) {
        const E* um = D + (long long)(m + 1) * stride;
        k_mr_set_spmv<<<1, 1, 0, s>>>(st, um, d_q);
        const int rc = launch_spmv<ROLE_GEN>(A, s);
        if (rc != MSOLVE_OK) return rc;
        k_mr_usub<E><<<grid, kThreads, 0, s>>>(st, D + (long long)m * stride, (const E*)d_q, um, n, m);
    }
    MSOLVE_CU(cudaGetLastError());
    return MSOLVE_OK;
}

template <typename E>
static int multirhs_finish(const msolve_matrix* A, void* d_x, int S, const char* d_slots, long long stride, const double* d_wtab, cudaStream_t s) {
    const long long n = A->dev.n;
    if (S < 2) return MSOLVE_OK;
    const int grid = (int)std::max(1ll, std::min<long long>((long long)A->num_sms * 4, (n + kThreads - 1) / kThreads));
    const E* U = (const E*)d_slots + stride;          // slot m+1 = u_m
    if (S <= 16) k_mr_add_guess16<E><<<grid, kThreads, 0, s>>>((E*)d_x, U, d_wtab, n, stride, S);
    else k_mr_add_guess<E><<<grid, kThreads, 0, s>>>((E*)d_x, U, d_wtab, n, stride, S);
    MSOLVE_CU(cudaGetLastError());
    return MSOLVE_OK;
}

}  // namespace msolve

using namespace msolve;

static size_t mr_align(size_t v) { return (v + 255) / 256 * 256; }

extern "C" size_t msolve_multirhs_workspace_bytes(const msolve_matrix* A, int nshifts, int algorithm) {
    const size_t base = msolve_workspace_bytes(A, nshifts, algorithm);
    if (!base) return 0;
    const size_t vb = mr_align((size_t)pk_stride_elems(A) * elem_bytes(A->dtype));
    return base + vb * (size_t)nshifts + mr_align(sizeof(double) * (size_t)nshifts * (size_t)nshifts) + 256;
}

extern "C" int msolve_solve_multirhs(const msolve_matrix* A, int algorithm, const void* d_B, const double* h_shifts,
                                     int nshifts, double tol, int max_iter, void* d_x, void* d_workspace,
                                     size_t workspace_bytes, int* h_iterations, int* h_conv_iter, double* h_relres,
                                     void* stream_) {
    if (!A) return fail(MSOLVE_EINVAL, "msolve_solve_multirhs: A is NULL");
    if (algorithm != MSOLVE_ALG_CGM && algorithm != MSOLVE_ALG_BICGSTABM) return fail(MSOLVE_EINVAL, "msolve_solve_multirhs: bad algorithm");
    if (!d_B || !d_x || !h_shifts || !d_workspace) return fail(MSOLVE_EINVAL, "msolve_solve_multirhs: NULL argument");
    const size_t need = msolve_multirhs_workspace_bytes(A, nshifts, algorithm);
    if (!need) return fail(MSOLVE_EINVAL, "msolve_solve_multirhs: nshifts must be in [1, %d]", kMaxShifts);
    if (workspace_bytes < need) return fail(MSOLVE_ENOMEM, "msolve_solve_multirhs: workspace too small (%zu < %zu)", workspace_bytes, need);
    if (((uintptr_t)d_B & 15u) || ((uintptr_t)d_x & 15u)) return fail(MSOLVE_EINVAL, "msolve_solve_multirhs: d_B / d_x must be 16-byte aligned");
    if (!(tol >= 0.0) || max_iter < 0) return fail(MSOLVE_EINVAL, "msolve_solve_multirhs: bad tol / max_iter");
    for (int i = 0; i < nshifts; ++i)
        for (int j = 0; j < i; ++j)
            if (h_shifts[i] == h_shifts[j]) return fail(MSOLVE_EINVAL, "msolve_solve_multirhs: shifts %d and %d are equal (the construction needs pairwise distinct shifts)", j, i);
    int rc = check_device(A, "msolve_solve_multirhs");
    if (rc != MSOLVE_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t base = msolve_workspace_bytes(A, nshifts, algorithm);
    const size_t vb = mr_align((size_t)pk_stride_elems(A) * elem_bytes(A->dtype));
    char* ws = (char*)mr_align((size_t)(uintptr_t)d_workspace);
    char* d_slots = ws + mr_align(base);
    double* d_wtab = (double*)(d_slots + vb * (size_t)nshifts);
    const long long stride_e = (long long)(vb / elem_bytes(A->dtype));
    if (A->dev.n == 0) return run_solver(algorithm, A, d_B, h_shifts, nshifts, tol, max_iter, d_x, ws, base, h_iterations, h_conv_iter, h_relres, stream_, 0);
    SigmaArg sg;
    for (int k = 0; k < kMaxShifts; ++k) sg.v[k] = k < nshifts ? h_shifts[k] : 0.0;
    k_mr_set_sigma<<<1, 128, 0, stream>>>(A->d_state, sg, nshifts);
    void* d_q = ws + 2 * vb;                               // the solver's q vector: free until the solve starts
    switch (A->dtype) {
        case MSOLVE_C128: rc = multirhs_setup<double2>(A, d_B, nshifts, d_slots, stride_e, d_wtab, d_q, stream); break;
        case MSOLVE_C64:  rc = multirhs_setup<float2>(A, d_B, nshifts, d_slots, stride_e, d_wtab, d_q, stream); break;
        case MSOLVE_F64:  rc = multirhs_setup<double>(A, d_B, nshifts, d_slots, stride_e, d_wtab, d_q, stream); break;
        default:          rc = multirhs_setup<float>(A, d_B, nshifts, d_slots, stride_e, d_wtab, d_q, stream); break;
    }
    if (rc != MSOLVE_OK) return rc;
    // slot 0 = r0: the common right-hand side of the multishift solve; thresholds tol ||b_i|| (rhs_norm on the device)
    const int status = run_solver(algorithm, A, d_slots, h_shifts, nshifts, tol, max_iter, d_x, ws, base, h_iterations,
                                  h_conv_iter, h_relres, stream_, 1);
    if (status < 0) return status;
    const int64_t solver_launches = A->last_launches;
    switch (A->dtype) {
        case MSOLVE_C128: rc = multirhs_finish<double2>(A, d_x, nshifts, d_slots, stride_e, d_wtab, stream); break;
        case MSOLVE_C64:  rc = multirhs_finish<float2>(A, d_x, nshifts, d_slots, stride_e, d_wtab, stream); break;
        case MSOLVE_F64:  rc = multirhs_finish<double>(A, d_x, nshifts, d_slots, stride_e, d_wtab, stream); break;
        default:          rc = multirhs_finish<float>(A, d_x, nshifts, d_slots, stride_e, d_wtab, stream); break;
    }
    if (rc != MSOLVE_OK) return rc;
    MSOLVE_CU(cudaStreamSynchronize(stream));
    const int setup = 3 + (nshifts <= 16 ? 1 : nshifts) + (nshifts - 1) * (2 + spmv_launches(A));
    const_cast<msolve_matrix*>(A)->last_launches = solver_launches + setup + (nshifts >= 2 ? 1 : 0);
    return status;
}
