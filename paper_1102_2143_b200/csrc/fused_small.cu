// fused_small.cu -- the WHOLE solve as one cooperative kernel, for systems whose matrix and vectors live in L2
// (BASELINE configs 1-2: 31 KB and 16.5 MB per iteration).  There the iteration as a graph of 5 (CG-M) / 7
// (BiCGStab-M) kernels is bound by launch latency, not by bytes (SURVEY.md section 7 "tiny configs are
// launch-latency bound": config 2 spends 24.6 us per iteration on 2.7 us of traffic).  Here one persistent grid
// (one CTA per SM at most, launched cooperatively so that all CTAs are resident) runs init and every iteration, with
// a grid-wide barrier wherever the graph path has a kernel boundary that carries a dependency across rows; a barrier
// that follows a reducing step carries the sum with it (fused_allreduce):
//   CG-M       p <- r + alpha p | SpMV + <p,Ap> | scalars #1, fused multishift update + |r|^2 | scalars #2      (3 barriers)
//   BiCGStab-M SpMV#1 + <r0,q> | scalars, s <- r + beta q | SpMV#2 + dots | scalars, fused update | scalars    (4 barriers)
// The steps are the SAME device functions the graph path runs as separate kernels (kernels.cuh, spmv.cuh row
// bodies).  Every CTA keeps its own copy of the recurrence scalars in shared memory and runs the scalar steps
// redundantly on the fixed-order sum of the per-CTA partials, so no CTA ever waits for a scalar another one
// computes, and the results are bit-reproducible for a given grid.  Alg. 1 step for step.
#include "handle.h"
#include "tuning.h"
#include "kernels.cuh"
#include "fused_sync.cuh"
#include "spmv.cuh"
#include "spmv_lattice.cuh"

namespace msolve {

constexpr int kFusedThreads = 512;
enum { FS_CSR2 = 2, FS_CSR4 = 4, FS_CSR8 = 8, FS_CSR32 = 32, FS_BSR3 = 100, FS_LAT = 101 };

template <typename E, int SEL, int ROLE>
__device__ __forceinline__ void fused_spmv(const MatDev& A, const SolveHeader& h, double* acc) {
    const E* x; E* y; const E* u;
    role_vectors_h<E, ROLE>(h, x, y, u);
    if constexpr (SEL == FS_BSR3) bsr3_rows_body<E, ROLE, false>(A, x, y, u, acc, blockIdx.x, gridDim.x);
    else if constexpr (SEL == FS_LAT) lat_rows_body<E, ROLE, false>(A, x, y, u, acc, blockIdx.x, gridDim.x);
    else csr_vector_body<E, SEL, ROLE, false, false>(A, x, y, u, acc, blockIdx.x, gridDim.x);
}

template <typename E, int VEC, int SEL>
__global__ void __launch_bounds__(kFusedThreads, 1) k_cgm_fused(MatDev A, SolveState* st, const __grid_constant__ SolveHeader hp) {
    extern __shared__ __align__(16) unsigned char dyn[];
    Recur& rc = *(Recur*)dyn;
    SolveResult& res = *(SolveResult*)(dyn + kFusedOffRes);
    const SolveHeader& h = *(const SolveHeader*)(dyn + kFusedOffHdr);
    double* rhs_norm = (double*)(dyn + kFusedOffNorm);
    __shared__ double red[kAccMax * 32];
    fused_stage_header(hp, st, dyn + kFusedOffHdr, rhs_norm);
    const int cta = blockIdx.x, ncta = gridDim.x;
    unsigned long long gen = st->fused_gen;                                           // written back by CTA 0 at the end
    double acc[1], s[1];
    acc[0] = init_vectors_fn<E, VEC>(h, cta, ncta);                                  // l.9-10, 13: r <- b, p <- b, <b,b>
    fused_allreduce<1>(st, gen, acc, s, red);
    init_state_fn(h, res, rc, s[0]);
    PhaseClock clk(h.phase_ns);
    while (!res.done) {
        if (res.n_iter > 0) {
            cgm_pupdate_fn<E, VEC>(h, rc, cta, ncta);                                 // l.27
            clk.mark(0);
            fused_allreduce<0>(st, gen, nullptr, nullptr, red);                       // p complete before it is gathered
            clk.mark(1);
        }
        acc[0] = 0.0;
        fused_spmv<E, SEL, ROLE_CG>(A, h, acc);                                       // l.18-19
        clk.mark(2);
        fused_allreduce<1>(st, gen, acc, s, red);
        clk.mark(3);
        cgm_scal1_fn(h, res, rc, s[0]);                                               // l.20, 22, 23
        if (res.done) break;                                                          // breakdown: the same in every CTA
        acc[0] = cgm_update_fn<E, VEC, kUnrollCgm, false>(h, res, rc, cta, ncta);            // l.21, 24, 28, 29
        clk.mark(4);
        fused_allreduce<1>(st, gen, acc, s, red);
        clk.mark(5);
        cgm_scal2_fn(h, res, rc, rhs_norm, s[0], cta == 0 ? h.hist : nullptr);   // l.25, 26, 30, 31, 15
    }
    if (clk.ns) clk.ns[15] += (unsigned long long)res.n_iter;
    fused_publish(st, res, gen);
}

template <typename E, int VEC, int SEL>
__global__ void __launch_bounds__(kFusedThreads, 1) k_bi_fused(MatDev A, SolveState* st, const __grid_constant__ SolveHeader hp) {
    extern __shared__ __align__(16) unsigned char dyn[];
    Recur& rc = *(Recur*)dyn;
    SolveResult& res = *(SolveResult*)(dyn + kFusedOffRes);
    const SolveHeader& h = *(const SolveHeader*)(dyn + kFusedOffHdr);
    double* rhs_norm = (double*)(dyn + kFusedOffNorm);
    __shared__ double red[kAccMax * 32];
    fused_stage_header(hp, st, dyn + kFusedOffHdr, rhs_norm);
    const int cta = blockIdx.x, ncta = gridDim.x;
    unsigned long long gen = st->fused_gen;
    double acc[5], s[5];
    acc[0] = init_vectors_fn<E, VEC>(h, cta, ncta);
    fused_allreduce<1>(st, gen, acc, s, red);
    init_state_fn(h, res, rc, s[0]);
    PhaseClock clk(h.phase_ns);
    while (!res.done) {
#pragma unroll
        for (int a = 0; a < 5; ++a) acc[a] = 0.0;
        fused_spmv<E, SEL, ROLE_B1>(A, h, acc);                                       // q = A p, <r0,q>
        clk.mark(0);
        fused_allreduce<2>(st, gen, acc, s, red);
        clk.mark(1);
        bi_scal1_fn(h, res, rc, zd{s[0], s[1]});
        if (res.done) break;
        bi_supdate_fn<E, VEC>(h, rc, cta, ncta);                                      // s = r + beta q
        clk.mark(2);
        fused_allreduce<0>(st, gen, nullptr, nullptr, red);                           // s complete before it is gathered
        clk.mark(3);
#pragma unroll
        for (int a = 0; a < 5; ++a) acc[a] = 0.0;
        fused_spmv<E, SEL, ROLE_B2>(A, h, acc);                                       // t = A s, <t,s>, <t,t>, <r0,t>
        clk.mark(4);
        fused_allreduce<5>(st, gen, acc, s, red);
        clk.mark(5);
        bi_scal2_fn(h, res, rc, s);
        if (res.done) break;
        acc[0] = bi_update_fn<E, VEC, kUnrollBi, false>(h, res, rc, cta, ncta);              // r', p, x_k, p_k, |r'|^2
        clk.mark(6);
        fused_allreduce<1>(st, gen, acc, s, red);                                     // also: p complete before SpMV#1
        clk.mark(7);
        bi_scal3_fn(h, res, rc, rhs_norm, s[0], cta == 0 ? h.hist : nullptr);
    }
    if (clk.ns) clk.ns[15] += (unsigned long long)res.n_iter;
    fused_publish(st, res, gen);
}

// ------------------------------------------------------------------------------------------- host side
static int fused_selector(const msolve_matrix* A) {
    if (A->format == FMT_BSR3) return FS_BSR3;
    if (A->format == FMT_LATTICE) return FS_LAT;
    if (A->format == FMT_CSR && A->kernel == KERNEL_VECTOR && (A->lanes == 2 || A->lanes == 4 || A->lanes == 8 || A->lanes == 32)) return A->lanes;
    return 0;
}

bool fused_supported(const msolve_matrix* A) {
    if (!fused_selector(A) || A->opt.update_kernel != 0 || A->opt.loop_mode != 0) return false;
    int coop = 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, A->device) != cudaSuccess || !coop) return false;
    return true;
}

template <typename K>
static int launch_coop(const msolve_matrix* A, K kernel, long long work_threads, cudaStream_t s) {
    const int smem = kFusedFixedBytes;
    int rc = ensure_smem(A, (const void*)kernel, smem);
    if (rc != MSOLVE_OK) return rc;
    int per_sm = 0;
    MSOLVE_CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kFusedThreads, smem));
    if (per_sm < 1) return fail(MSOLVE_ECUDA, "fused kernel does not fit on an SM");
    const long long need = (work_threads + kFusedThreads - 1) / kFusedThreads;
    const int cap = std::min(A->num_sms, kFusedMaxCtas);
    int grid = (int)std::max(1ll, std::min<long long>(cap, need));
    if (A->opt.fused_ctas > 0) grid = std::min(cap, A->opt.fused_ctas);
    MatDev dev = A->dev;
    SolveState* st = A->d_state;
    SolveHeader hdr = A->h_stage->h;
    void* args[3] = {&dev, &st, &hdr};
    MSOLVE_CU(cudaLaunchCooperativeKernel((const void*)kernel, dim3(grid), dim3(kFusedThreads), args, (size_t)smem, s));
    return MSOLVE_OK;
}

template <typename E, int VEC, int SEL>
static int launch_fused_sel(const msolve_matrix* A, int alg, cudaStream_t s) {
    // threads that have work in the widest phase: the SpMV rows (times the lanes per row)
    const long long lanes = SEL >= 100 ? 1 : SEL;
    const long long work = std::max<long long>(A->dev.n * lanes, 1);
    if (alg == MSOLVE_ALG_CGM) return launch_coop(A, k_cgm_fused<E, VEC, SEL>, work, s);
    return launch_coop(A, k_bi_fused<E, VEC, SEL>, work, s);
}

template <typename E, int VEC>
static int launch_fused_t(const msolve_matrix* A, int alg, cudaStream_t s) {
    switch (fused_selector(A)) {
        case FS_CSR2: return launch_fused_sel<E, VEC, FS_CSR2>(A, alg, s);
        case FS_CSR4: return launch_fused_sel<E, VEC, FS_CSR4>(A, alg, s);
        case FS_CSR8: return launch_fused_sel<E, VEC, FS_CSR8>(A, alg, s);
        case FS_CSR32: return launch_fused_sel<E, VEC, FS_CSR32>(A, alg, s);
        case FS_BSR3: if constexpr (sizeof(E) == 2 * sizeof(typename RealOf<E>::type)) return launch_fused_sel<E, VEC, FS_BSR3>(A, alg, s); break;
        case FS_LAT: if constexpr (sizeof(E) == 2 * sizeof(typename RealOf<E>::type)) return launch_fused_sel<E, VEC, FS_LAT>(A, alg, s); break;
        default: break;
    }
    return fail(MSOLVE_EINVAL, "fused path: unsupported matrix format");
}

int launch_fused(const msolve_matrix* A, int alg, cudaStream_t s) {
    const bool v16 = A->dev.n % (long long)(16 / elem_bytes(A->dtype)) == 0;
    switch (A->dtype) {
        case MSOLVE_C128: return launch_fused_t<double2, 1>(A, alg, s);
        case MSOLVE_C64:  return v16 ? launch_fused_t<float2, 2>(A, alg, s) : launch_fused_t<float2, 1>(A, alg, s);
        case MSOLVE_F64:  return v16 ? launch_fused_t<double, 2>(A, alg, s) : launch_fused_t<double, 1>(A, alg, s);
        default:          return v16 ? launch_fused_t<float, 4>(A, alg, s) : launch_fused_t<float, 1>(A, alg, s);
    }
}

}  // namespace msolve
