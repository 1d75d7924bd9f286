// spmv_role.cu -- launch code of every SpMV kernel for ONE role (compiled four times by build.py with
// -DMSOLVE_ROLE=0..3: ROLE_CG, ROLE_B1, ROLE_B2, ROLE_GEN; the fused reductions of Alg. 1 l.19,
// PAPER.md:111, and of the BiCGStab-M steps differ per role, the matrix traversal does not).
#include "handle.h"
#include "tuning.h"
#include "spmv.cuh"
#include "spmv_merge.cuh"
#include "spmv_csr_tile.cuh"
#include "spmv_lattice.cuh"

#ifndef MSOLVE_ROLE
#error "compile with -DMSOLVE_ROLE=0..3"
#endif

namespace msolve {

template <typename E> struct IsComplex { static constexpr bool value = false; };
template <> struct IsComplex<float2> { static constexpr bool value = true; };
template <> struct IsComplex<double2> { static constexpr bool value = true; };

static int merge_grid(const msolve_matrix* A, int cps) { return std::max(1, std::min(A->num_sms * cps, A->dev.aux_count)); }
static int merge_fixup_grid(const msolve_matrix* A) { return std::max(1, std::min(A->num_sms, (A->dev.aux_count + kThreads - 1) / kThreads)); }

template <typename T, int LANES, int U, int ROLE>
static int launch_csr_tile(const msolve_matrix* A, cudaStream_t s) {
    typedef CsrTile<T> P;
    typedef CsrTileCfg<T, LANES, U> Cfg;
    auto k = k_spmv_csr_tile<T, LANES, U, P::STAGES, P::CPS, ROLE>;
    const int smem = Cfg::smem_bytes(P::STAGES);
    const int rc = ensure_smem(A, (const void*)k, smem);
    if (rc != MSOLVE_OK) return rc;
    const long long ntiles = (A->dev.n + Cfg::kRows - 1) / Cfg::kRows;
    const int grid = (int)std::max(1ll, std::min<long long>((long long)A->num_sms * P::CPS, ntiles));
    k<<<grid, Cfg::kThreadsTotal, smem, s>>>(A->dev, A->d_state);
    return MSOLVE_OK;
}

// the blocked kernel's geometry: 4-D, x0-rows of 32 sites (lane = x0), extents the block divides
template <typename T>
static bool lat_blk_supported(const msolve_matrix* A) {
    if constexpr (sizeof(T) == 2 * sizeof(typename RealOf<T>::type)) {
        typedef LatBlkTile<T> B;
        const MatDev& d = A->dev;
        return d.lat_ndim == 4 && d.lat_ext[0] == 32 && d.lat_ext[1] % B::R1 == 0 && d.lat_ext[2] % B::R2 == 0;
    }
    return false;
}

// which lattice tile kernel this launch takes (1 = (term, site), 2 = warp per tile, 3 = hybrid, 4 = blocked)
template <typename T, int ROLE>
static int lattice_choice(const msolve_matrix* A) {
    // 4-D lattices with x0-rows of 32 sites take the blocked kernel: config 4 complex64 0.148 -> 0.121 ms against
    // the warp kernel, complex128 0.241 -> 0.240 ms against the hybrid one, second BiCGStab-M SpMV 0.287 -> 0.270 ms
    if ((A->opt.lattice_kernel == 4 || A->opt.lattice_kernel == 0) && lat_blk_supported<T>(A)) return 4;
    if (A->opt.lattice_kernel != 0 && A->opt.lattice_kernel != 4) return A->opt.lattice_kernel;
    // the second BiCGStab-M SpMV (five accumulators, two extra operands) spills in the hybrid kernel at 255
    // registers (config3x: spmv2_dots 0.278 ms all-TMA, 0.320 ms hybrid): it stays on the all-TMA kernels
    if (ROLE == ROLE_B2 && LatDefault<T>::kernel == 3) return sizeof(T) == 16 ? 1 : 2;
    return LatDefault<T>::kernel;
}

// MSOLVE_CFG_X_WINDOW: the launch carries an L2 access-policy window over the gathered vector (persisting hits,
// streaming misses), so that the matrix stream does not evict x from L2; the load instructions are unchanged.
// The window is a launch attribute: captured into the graph's kernel node, hence the graph is re-captured when
// the vector moves (LoopGraph::xptr).
template <int ROLE, typename K>
static int launch_with_x_window(const msolve_matrix* A, K k, int grid, int threads, cudaStream_t s) {
    const SolveHeader& h = A->h_stage->h;
    const void* xptr = ROLE == ROLE_GEN ? h.sp_x : ROLE == ROLE_B2 ? h.s : h.p;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)threads); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeAccessPolicyWindow;
    cudaAccessPolicyWindow& w = attr[0].val.accessPolicyWindow;
    w.base_ptr = const_cast<void*>(xptr);
    w.num_bytes = std::min((size_t)A->dev.n * elem_bytes(A->dtype), A->l2_window_max);
    w.hitRatio = (float)std::min(1.0, (double)A->l2_persist_bytes / (double)std::max<size_t>(w.num_bytes, 1));
    w.hitProp = cudaAccessPropertyPersisting;
    w.missProp = cudaAccessPropertyStreaming;
    cfg.attrs = attr; cfg.numAttrs = 1;
    MSOLVE_CU(cudaLaunchKernelEx(&cfg, k, A->dev, A->d_state));
    return MSOLVE_OK;
}

template <typename T, int ROLE>
static int launch_spmv_t(const msolve_matrix* A, cudaStream_t s) {
    int rc;
    if (A->format == FMT_CSR && A->kernel == KERNEL_CSR_TILE) {
        if (sizeof(T) == 16 || A->tile_u == 4) {
            switch (A->lanes) {
                case 2: return launch_csr_tile<T, 2, 4, ROLE>(A, s);
                case 4: return launch_csr_tile<T, 4, 4, ROLE>(A, s);
                case 8: if constexpr (sizeof(T) == 16) return launch_csr_tile<T, 8, 4, ROLE>(A, s); break;
                default: if constexpr (sizeof(T) == 16) return launch_csr_tile<T, 16, 4, ROLE>(A, s); break;
            }
        } else if constexpr (sizeof(T) < 16) {
            switch (A->lanes) {
                case 4: return launch_csr_tile<T, 4, 8, ROLE>(A, s);
                case 8: return launch_csr_tile<T, 8, 8, ROLE>(A, s);
                default: return launch_csr_tile<T, 16, 8, ROLE>(A, s);
            }
        }
        return fail(MSOLVE_EINVAL, "spmv: no TMA-staged vector-CSR shape for %d lanes", A->lanes);
    }
    if (A->format == FMT_CSR && A->kernel == KERNEL_MERGE) {
        typedef MergeTile<T> M;
        auto kp = k_spmv_csr_merge<T, M::CAP, M::STAGES, M::CPS, ROLE, true>;     // x pinned in L2
        auto kn = k_spmv_csr_merge<T, M::CAP, M::STAGES, M::CPS, ROLE, false>;
        const int smem = MergeCfg<T, M::CAP>::smem_bytes(M::STAGES);
        if ((rc = ensure_smem(A, (const void*)kp, smem)) != MSOLVE_OK) return rc;
        if ((rc = ensure_smem(A, (const void*)kn, smem)) != MSOLVE_OK) return rc;
        const int grid = merge_grid(A, M::CPS);
        (A->dev.x_pin ? kp : kn)<<<grid, MergeCfg<T, M::CAP>::kThreadsTotal, smem, s>>>(A->dev, A->d_state);
        k_spmv_csr_merge_fixup<T, ROLE><<<merge_fixup_grid(A), kThreads, 0, s>>>(A->dev, A->d_state, grid);
        return MSOLVE_OK;
    }
    if constexpr (IsComplex<T>::value) {               // BSR3 / lattice = SU(3) blocks: complex only
        if (A->format == FMT_BSR3 && A->kernel == KERNEL_BSR_TMA) {
            typedef BsrTile<T> B;
            constexpr int CPS = B::CPS - (ROLE == ROLE_B2 ? kBsrCpsLessB2 : 0);
            auto k = k_spmv_bsr3_tma<T, B::TB, B::STAGES, CPS, ROLE>;
            const int smem = BsrTmaCfg<T, B::TB>::smem_bytes(B::STAGES);
            if ((rc = ensure_smem(A, (const void*)k, smem)) != MSOLVE_OK) return rc;
            const int grid = std::max(1, std::min(A->num_sms * CPS, A->dev.aux_count));
            k<<<grid, BsrTmaCfg<T, B::TB>::kThreadsTotal, smem, s>>>(A->dev, A->d_state);
            return MSOLVE_OK;
        }
        if (A->format == FMT_LATTICE && A->kernel == KERNEL_LAT_TMA) {
            const int which = lattice_choice<T, ROLE>(A);
            if (which == 4) {
                typedef LatBlkTile<T> B;
                typedef LatBlkCfg<T, B::R1, B::R2, B::STAGES> Cfg;
                auto k = k_spmv_lat_blk<T, B::R1, B::R2, B::STAGES, ROLE>;
                if ((rc = ensure_smem(A, (const void*)k, Cfg::smem_bytes())) != MSOLVE_OK) return rc;
                const long long ntiles = (long long)(A->dev.lat_ext[1] / B::R1) * (A->dev.lat_ext[2] / B::R2) * A->dev.lat_ext[3];
                const int grid = (int)std::max(1ll, std::min<long long>(A->num_sms, ntiles));
                k<<<grid, Cfg::kThreadsTotal, Cfg::smem_bytes(), s>>>(A->dev, A->d_state);
                return MSOLVE_OK;
            }
            if (which == 3) {
                typedef LatHybTile<T> H;
                auto k = k_spmv_lat_hyb<T, H::W, H::STAGES, ROLE>;
                const int smem = LatHybCfg<T, H::W>::smem_bytes(H::STAGES);
                if ((rc = ensure_smem(A, (const void*)k, smem)) != MSOLVE_OK) return rc;
                const int grid = std::max(1, std::min(A->num_sms, A->dev.aux_count));
                k<<<grid, LatHybCfg<T, H::W>::kThreadsTotal, smem, s>>>(A->dev, A->d_state);
                return MSOLVE_OK;
            }
            if (which == 2) {
                typedef LatWarpTile<T> L;
                auto k = k_spmv_lat_warp<T, L::W, kLatWarpProducers, L::STAGES, ROLE>;
                const int smem = LatWarpCfg<T, L::W, kLatWarpProducers>::smem_bytes(L::STAGES);
                if ((rc = ensure_smem(A, (const void*)k, smem)) != MSOLVE_OK) return rc;
                const int grid = std::max(1, std::min(A->num_sms, A->dev.aux_count));
                k<<<grid, LatWarpCfg<T, L::W, kLatWarpProducers>::kThreadsTotal, smem, s>>>(A->dev, A->d_state);
                return MSOLVE_OK;
            }
            typedef LatTile<T> L;
            auto k = k_spmv_lat_tma<T, L::NS, L::STAGES, L::CPS, ROLE>;
            const int smem = LatCfg<T, L::NS>::smem_bytes(L::STAGES);
            if ((rc = ensure_smem(A, (const void*)k, smem)) != MSOLVE_OK) return rc;
            const int grid = std::max(1, std::min(A->num_sms * L::CPS, A->dev.aux_count));
            k<<<grid, LatCfg<T, L::NS>::kThreadsTotal, smem, s>>>(A->dev, A->d_state);
            return MSOLVE_OK;
        }
        if (A->format == FMT_LATTICE) {
            auto k = k_spmv_lat_rows<T, ROLE>;
            k<<<grid_for(A, k, A->dev.n, kThreads), kThreads, 0, s>>>(A->dev, A->d_state);
            return MSOLVE_OK;
        }
        if (A->format == FMT_BSR3) {
            auto k = k_spmv_bsr3_rows<T, ROLE>;
            k<<<grid_for(A, k, A->dev.n, kThreads), kThreads, 0, s>>>(A->dev, A->d_state);
            return MSOLVE_OK;
        }
    }
#define VEC_CASE(L)                                                                                     \
    case L: {                                                                                           \
        auto k = A->dev.x_pin ? k_spmv_csr_vector<T, L, ROLE, true> : k_spmv_csr_vector<T, L, ROLE, false>; \
        const int grid = grid_for(A, k, A->dev.n, kThreads / L);                                        \
        if (A->opt.x_window) return launch_with_x_window<ROLE>(A, k, grid, kThreads, s);                \
        k<<<grid, kThreads, 0, s>>>(A->dev, A->d_state);                                                \
        return MSOLVE_OK;                                                                               \
    }
    switch (A->lanes) {
        VEC_CASE(2) VEC_CASE(4) VEC_CASE(8) VEC_CASE(16) VEC_CASE(32)
        default: break;
    }
#undef VEC_CASE
    return fail(MSOLVE_EINVAL, "spmv: no kernel for format %d / %d lanes", A->format, A->lanes);
}

template <>
int launch_spmv<MSOLVE_ROLE>(const msolve_matrix* A, cudaStream_t s) {
    switch (A->dtype) {
        case MSOLVE_C128: return launch_spmv_t<double2, MSOLVE_ROLE>(A, s);
        case MSOLVE_C64:  return launch_spmv_t<float2, MSOLVE_ROLE>(A, s);
        case MSOLVE_F64:  return launch_spmv_t<double, MSOLVE_ROLE>(A, s);
        default:          return launch_spmv_t<float, MSOLVE_ROLE>(A, s);
    }
}

}  // namespace msolve
