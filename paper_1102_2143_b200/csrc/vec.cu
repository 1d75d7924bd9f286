// vec.cu -- launch code of the vector-update and scalar-recurrence kernels (kernels.cuh, update_tma.cuh):
// SURVEY.md 8(a) rows A1, A4, A5, A6 (CG-M, Alg. 1 l.20-31) and the BiCGStab-M analogues.
#include "handle.h"
#include "tuning.h"
#include "kernels.cuh"
#include "update_tma.cuh"

namespace msolve {

// ---- the one-CTA scalar kernels: fixed-order sum of the per-CTA partials, then the recurrence step (kernels.cuh).
// `cond` is the WHILE node's handle (use_cond = 0 in chunked mode).
__global__ void __launch_bounds__(kThreads) k_init_state(SolveState* st) {
    __shared__ double red[32];
    double s[1];
    reduce_partials<1>(st, s, red);
    init_state_fn(st->h, st->res, st->rc, s[0]);
    if (st->h.defer) defer_init(st->df);
}

__global__ void __launch_bounds__(kThreads) k_cgm_scal1(SolveState* st) {
    if (st->res.done) return;
    __shared__ double red[32];
    double s[1];
    reduce_partials<1>(st, s, red);
    cgm_scal1_fn(st->h, st->res, st->rc, s[0]);
    if (st->h.defer) cgm_defer_coef_fn(st->h, st->res, st->rc, st->df);
}

__global__ void __launch_bounds__(kThreads) k_cgm_scal2(SolveState* st, cudaGraphConditionalHandle cond, int use_cond) {
    if (st->res.done) { if (use_cond && threadIdx.x == 0) cudaGraphSetConditional(cond, 0); return; }
    __shared__ double red[32];
    double s[1];
    reduce_partials<1>(st, s, red);
    cgm_scal2_fn(st->h, st->res, st->rc, st->rhs_norm, s[0], st->h.hist);
    if (st->h.defer) cgm_defer_advance(st->h, st->df);
    if (use_cond && threadIdx.x == 0) cudaGraphSetConditional(cond, st->res.done ? 0u : 1u);
}

__global__ void __launch_bounds__(kThreads) k_bi_scal1(SolveState* st) {
    if (st->res.done) return;
    __shared__ double red[2 * 32];
    double s[2];
    reduce_partials<2>(st, s, red);
    bi_scal1_fn(st->h, st->res, st->rc, zd{s[0], s[1]});
}

__global__ void __launch_bounds__(kThreads) k_bi_scal2(SolveState* st) {
    if (st->res.done) return;
    __shared__ double red[5 * 32];
    double s[5];
    reduce_partials<5>(st, s, red);
    bi_scal2_fn(st->h, st->res, st->rc, s);
}

__global__ void __launch_bounds__(kThreads) k_bi_scal3(SolveState* st, cudaGraphConditionalHandle cond, int use_cond) {
    if (st->res.done) { if (use_cond && threadIdx.x == 0) cudaGraphSetConditional(cond, 0); return; }
    __shared__ double red[32];
    double s[1];
    reduce_partials<1>(st, s, red);
    bi_scal3_fn(st->h, st->res, st->rc, st->rhs_norm, s[0], st->h.hist);
    if (use_cond && threadIdx.x == 0) cudaGraphSetConditional(cond, st->res.done ? 0u : 1u);
}

// element-wise kernels: 16 bytes (1, 2 or 4 elements) per access when the length allows it
static bool vec16(const msolve_matrix* A) {
    const long long m = (long long)(16 / elem_bytes(A->dtype));
    return A->dev.n % m == 0 && A->x_stride % m == 0;
}

#define DISPATCH_VEC(A, KERNEL, ...)                                                       \
    do {                                                                                   \
        const bool v16_ = vec16(A);                                                        \
        switch ((A)->dtype) {                                                              \
            case MSOLVE_C128: KERNEL(double2, 1, __VA_ARGS__); break;                      \
            case MSOLVE_C64: if (v16_) { KERNEL(float2, 2, __VA_ARGS__); } else { KERNEL(float2, 1, __VA_ARGS__); } break; \
            case MSOLVE_F64: if (v16_) { KERNEL(double, 2, __VA_ARGS__); } else { KERNEL(double, 1, __VA_ARGS__); } break; \
            default:         if (v16_) { KERNEL(float, 4, __VA_ARGS__); } else { KERNEL(float, 1, __VA_ARGS__); } break;   \
        }                                                                                  \
    } while (0)

// grid of the flush kernel: resident CTAs per SM with its dynamic shared memory, capped by the work
static int flush_grid(const msolve_matrix* A, const void* k, int smem, long long work) {
    if (A->flush_ctas_per_sm < 1) {            // once per handle (one element type and pack width per handle)
        int per_sm = 1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, kThreads, (size_t)smem) != cudaSuccess || per_sm < 1) per_sm = 1;
        A->flush_ctas_per_sm = per_sm;
    }
    const long long need = (work + kThreads - 1) / kThreads;
    return (int)std::max(1ll, std::min<long long>((long long)A->num_sms * A->flush_ctas_per_sm, need));
}

template <typename T>
static int launch_cgm_update_tma(const msolve_matrix* A, cudaStream_t s) {
    typedef UpdTmaCfg<T> U;
    auto k = k_cgm_update_tma<T, kUpdStages, kUpdLag>;
    const int smem = U::smem_bytes(kUpdStages);
    const int rc = ensure_smem(A, (const void*)k, smem);
    if (rc != MSOLVE_OK) return rc;
    const long long ntiles = (A->dev.n / U::VEC + U::kTile - 1) / U::kTile;
    const int grid = (int)std::max(1ll, std::min<long long>(A->num_sms, ntiles));
    k<<<grid, U::kThreadsTotal, smem, s>>>(A->d_state);
    return MSOLVE_OK;
}

#define L_INIT(T, V, A, s) { auto k = k_init_vectors<T, V>; k<<<grid_for(A, k, (A)->dev.n / V, kThreads * 4), kThreads, 0, s>>>((A)->d_state); }
#define L_PUPD(T, V, A, s) { auto k = k_cgm_pupdate<T, V>; k<<<grid_for(A, k, (A)->dev.n / V, kThreads * 4), kThreads, 0, s>>>((A)->d_state); }
#define L_CUPD(T, V, A, s) {                                                                            \
    if (V * sizeof(T) == 16 && (A)->opt.update_kernel == 1) rc = launch_cgm_update_tma<T>(A, s);           \
    else { auto k = k_cgm_update<T, V, kUnrollCgm>; k<<<grid_for(A, k, (A)->dev.n / V, kThreads), kThreads, 0, s>>>((A)->d_state); } }
#define L_RUPD(T, V, A, s) { auto k = k_cgm_rupdate<T, V>; k<<<grid_for(A, k, (A)->dev.n / V, kThreads * 4), kThreads, 0, s>>>((A)->d_state); }
#define L_FLSH(T, V, A, s) {                                                                            \
    auto k = k_cgm_flush<T, V, kUnrollFlush>;                                                           \
    const int smem = 2 * kMaxShifts * kDeferMax * (int)sizeof(typename RealOf<T>::type);                \
    rc = ensure_smem(A, (const void*)k, smem);                                                          \
    if (rc == MSOLVE_OK) k<<<flush_grid(A, (const void*)k, smem, (A)->dev.n / V), kThreads, smem, s>>>((A)->d_state); }
#define L_SUPD(T, V, A, s) { auto k = k_bi_supdate<T, V>; k<<<grid_for(A, k, (A)->dev.n / V, kThreads * 4), kThreads, 0, s>>>((A)->d_state); }
#define L_BUPD(T, V, A, s) { auto k = k_bi_update<T, V, kUnrollBi>; k<<<grid_for(A, k, (A)->dev.n / V, kThreads), kThreads, 0, s>>>((A)->d_state); }

int launch_vec_kernel(const msolve_matrix* A, int alg, int j, cudaStream_t s, cudaGraphConditionalHandle cond, int use_cond) {
    SolveState* st = A->d_state;
    int rc = MSOLVE_OK;
    if (alg == MSOLVE_ALG_CGM) {
        switch (j) {
            case 0: DISPATCH_VEC(A, L_PUPD, A, s); break;
            case 2: k_cgm_scal1<<<1, kThreads, 0, s>>>(st); break;
            case 3: if (defer_len(A, alg) > 0) { DISPATCH_VEC(A, L_RUPD, A, s); } else { DISPATCH_VEC(A, L_CUPD, A, s); } break;
            case 4: k_cgm_scal2<<<1, kThreads, 0, s>>>(st, cond, use_cond); break;
            case 5: DISPATCH_VEC(A, L_FLSH, A, s); break;                    // deferred update only (kernels_per_iter)
            default: return fail(MSOLVE_EINVAL, "launch_vec_kernel: CG-M kernel %d is not a vector kernel", j);
        }
    } else {
        switch (j) {
            case 1: k_bi_scal1<<<1, kThreads, 0, s>>>(st); break;
            case 2: DISPATCH_VEC(A, L_SUPD, A, s); break;
            case 4: k_bi_scal2<<<1, kThreads, 0, s>>>(st); break;
            case 5: DISPATCH_VEC(A, L_BUPD, A, s); break;
            case 6: k_bi_scal3<<<1, kThreads, 0, s>>>(st, cond, use_cond); break;
            default: return fail(MSOLVE_EINVAL, "launch_vec_kernel: BiCGStab-M kernel %d is not a vector kernel", j);
        }
    }
    return rc;
}

int launch_init_vectors(const msolve_matrix* A, cudaStream_t s) {
    DISPATCH_VEC(A, L_INIT, A, s);
    return MSOLVE_OK;
}
int launch_init_state(const msolve_matrix* A, cudaStream_t s) {
    k_init_state<<<1, kThreads, 0, s>>>(A->d_state);
    return MSOLVE_OK;
}
int launch_init(const msolve_matrix* A, cudaStream_t s) {
    launch_init_vectors(A, s);
    return launch_init_state(A, s);
}

}  // namespace msolve
