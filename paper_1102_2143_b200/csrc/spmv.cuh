// spmv.cuh -- complex SpMV kernels with the dot products of the iteration fused into the
// epilogue (Alg. 1 l.18-19).
//
// Every kernel is persistent (grid = a multiple of the SM count, grid-stride over row tiles),
// streams the matrix with evict-first loads so that the gathered vector stays in the 126 MB L2,
// and writes ONE partial sum per CTA per reduced quantity; the partials are summed in fixed
// order by the scalar kernels (deterministic, no atomics on doubles).
//
// ROLE selects the vectors (read from the device-resident SolveState) and the fused reductions:
//   ROLE_CG  : y=q=A p,            acc[0]      = Re <p,q>                      (CG-M, l.19)
//   ROLE_B1  : y=q=A p,            acc[0..1]   = <r0,q>                        (BiCGStab-M)
//   ROLE_B2  : y=t=A s,            acc[0..1]   = <t,s>, acc[2] = <t,t>, acc[3..4] = <r0,t>
//   ROLE_GEN : y=sp_y=A sp_x,      acc[0..1]   = <sp_u, y>                     (msolve_spmv)
#pragma once

#include "common.cuh"

namespace msolve {

template <int ROLE> struct RoleAcc { static constexpr int value = ROLE == ROLE_CG ? 1 : (ROLE == ROLE_B2 ? 5 : 2); };

template <typename C, int ROLE>
__device__ __forceinline__ void role_vectors_h(const SolveHeader& h, const C*& x, C*& y, const C*& u) {
    if (ROLE == ROLE_CG)  { x = (const C*)h.p; y = (C*)h.q; u = nullptr; }
    if (ROLE == ROLE_B1)  { x = (const C*)h.p; y = (C*)h.q; u = (const C*)h.b; }
    if (ROLE == ROLE_B2)  { x = (const C*)h.s; y = (C*)h.t; u = (const C*)h.b; }
    if (ROLE == ROLE_GEN) { x = (const C*)h.sp_x; y = (C*)h.sp_y; u = (const C*)h.sp_u; }
}
template <typename C, int ROLE>
__device__ __forceinline__ void role_vectors(const SolveState* st, const C*& x, C*& y, const C*& u) {
    role_vectors_h<C, ROLE>(st->h, x, y, u);
}

// Fused reductions for one finished row (all accumulation in fp64, R14).
template <typename C, int ROLE>
__device__ __forceinline__ void role_epilogue(double* acc, long long row, C yi, const C* x, const C* u) {
    if (ROLE == ROLE_CG) {
        acc[0] += cdot_re(x[row], yi);                          // Re <p,q>
    } else if (ROLE == ROLE_B1 || ROLE == ROLE_GEN) {
        const C ui = u[row];
        acc[0] += cdot_re(ui, yi);                              // conj(u) y
        acc[1] += cdot_im(ui, yi);
    } else {
        const C xi = x[row];
        const C ui = u[row];
        acc[0] += cdot_re(yi, xi);                              // conj(y) x  = <t,s>
        acc[1] += cdot_im(yi, xi);
        acc[2] += cnorm2(yi);                                   // <t,t>
        acc[3] += cdot_re(ui, yi);                              // <r0,t>
        acc[4] += cdot_im(ui, yi);
    }
}

template <int NACC>
__device__ __forceinline__ void write_partials(SolveState* st, double (&acc)[NACC]) {
    __shared__ double red[NACC * 32];
    block_sum<NACC>(acc, red);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int a = 0; a < NACC; ++a) st->partial[a * kMaxPartials + blockIdx.x] = acc[a];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

// ------------------------------------------------------------------------------------------
// Vector-CSR: LANES lanes per row (LANES | 32), rows of a warp are consecutive, the lanes of a
// row read consecutive non-zeros (coalesced 16-byte values, 4-byte indices).  For short regular
// lattice rows (27 nnz: LANES = 8, four passes).
// ------------------------------------------------------------------------------------------
// NC = false: the gathered vector was written earlier in the SAME kernel launch (fused_small.cuh), so it must not go
// through the non-coherent load path; the matrix arrays always may.
template <typename E, int LANES, int ROLE, bool PIN, bool NC = true>
__device__ __forceinline__ void csr_vector_body(const MatDev& A, const E* x, E* y, const E* u, double* acc, int cta, int ncta) {
    typedef E C;
    const C* __restrict__ val = (const C*)A.val;
    const int32_t* __restrict__ colidx = A.colidx;
    const int32_t* __restrict__ rowptr = A.rowptr;
    constexpr int RPW = 32 / LANES;  // rows per warp
    constexpr bool HINT = sizeof(E) <= 8;
    const uint64_t polx = policy_evict_last(), polm = policy_evict_first();
    const int lane = threadIdx.x & 31;
    const int sub = lane % LANES;
    const long long warp = ((long long)cta * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)ncta * blockDim.x) >> 5;
    for (long long base = warp * RPW; base < A.n; base += nwarps * RPW) {
        const long long row = base + lane / LANES;
        const bool valid = row < A.n;
        int j = 0, e = 0;
        if (valid) { j = rowptr[row] + sub; e = rowptr[row + 1]; }
        C sum = cmake<C>(0.0, 0.0);
        // Long rows: the loads of a lane batched by kind (8 indices + 8 values, then the 8 gathers they address, then
        // the arithmetic); the rest one at a time.  What matters more is the register budget: at 6 CTAs per SM
        // (__launch_bounds__ below: 40 registers) config 5 complex128 runs at 1.20 ms, at the 34 registers ptxas
        // picks on its own the loads of the unrolled loop share registers and serialise: 1.43 ms
        // (profiles/r02_sweeps.md section 4).
        constexpr int UB = 8;
        for (; j + (UB - 1) * LANES < e; j += UB * LANES) {
            int c[UB];
            C v[UB], xv[UB];
#pragma unroll
            for (int t = 0; t < UB; ++t) { c[t] = ld_mat<HINT>(colidx + j + t * LANES, polm); v[t] = ld_mat<HINT>(val + j + t * LANES, polm); }
#pragma unroll
            for (int t = 0; t < UB; ++t) xv[t] = NC ? ld_xg<PIN>(x + c[t], polx) : x[c[t]];
#pragma unroll
            for (int t = 0; t < UB; ++t) sum = cfma(v[t], xv[t], sum);
        }
        for (; j < e; j += LANES) {
            const int c = ld_mat<HINT>(colidx + j, polm);
            const C v = ld_mat<HINT>(val + j, polm);
            sum = cfma(v, NC ? ld_xg<PIN>(x + c, polx) : x[c], sum);
        }
#pragma unroll
        for (int o = LANES / 2; o > 0; o >>= 1) sum = cshfl_xor_add(sum, o);
        if (valid && sub == 0) {
            y[row] = sum;
            role_epilogue<C, ROLE>(acc, row, sum, x, u);
        }
    }
}

template <typename E, int LANES, int ROLE, bool PIN>
__global__ void __launch_bounds__(kThreads, ROLE == ROLE_B2 ? 5 : 6) k_spmv_csr_vector(MatDev A, SolveState* st) {
    typedef E C;
    constexpr int NACC = RoleAcc<ROLE>::value;
    if (ROLE != ROLE_GEN && st->res.done) return;
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    csr_vector_body<E, LANES, ROLE, PIN>(A, x, y, u, acc, blockIdx.x, gridDim.x);
    write_partials<NACC>(st, acc);
}

// ------------------------------------------------------------------------------------------
// BSR3, one thread per scalar row (first, simple variant): thread (br, r) walks the blocks of
// block row br and multiplies row r of every 3x3 block with the 3-vector x[3*bcol .. +3].
// The three threads of a block row read one contiguous 144-byte (c128) block between them.
// ------------------------------------------------------------------------------------------
template <typename E, int ROLE, bool NC = true>
__device__ __forceinline__ void bsr3_rows_body(const MatDev& A, const E* x, E* y, const E* u, double* acc, int cta, int ncta) {
    typedef E C;
    const C* __restrict__ val = (const C*)A.val;
    const int32_t* __restrict__ bcol = A.colidx;
    const int32_t* __restrict__ browptr = A.rowptr;
    const long long stride = (long long)ncta * blockDim.x;
    const bool keep = A.mat_keep > 0;            // MSOLVE_CFG_MATRIX_L2_KEEP_PERCENT: hinted loads (policy_matrix)
    const uint64_t polm = policy_matrix(A.mat_keep);
    for (long long row = (long long)cta * blockDim.x + threadIdx.x; row < A.n; row += stride) {
        const long long br = row / 3;
        const int rr = (int)(row - 3 * br);
        const int jb = browptr[br], je = browptr[br + 1];
        C sum = cmake<C>(0.0, 0.0);
#pragma unroll 3
        for (int j = jb; j < je; ++j) {
            const C* blk = val + (long long)j * 9 + rr * 3;
            const C* xv = x + 3ll * bcol[j];
            const C a0 = keep ? ld_xg<true>(blk, polm) : ld_stream(blk);
            const C a1 = keep ? ld_xg<true>(blk + 1, polm) : ld_stream(blk + 1);
            const C a2 = keep ? ld_xg<true>(blk + 2, polm) : ld_stream(blk + 2);
            sum = cfma(a0, NC ? ld_ro(xv) : xv[0], sum);
            sum = cfma(a1, NC ? ld_ro(xv + 1) : xv[1], sum);
            sum = cfma(a2, NC ? ld_ro(xv + 2) : xv[2], sum);
        }
        y[row] = sum;
        role_epilogue<C, ROLE>(acc, row, sum, x, u);
    }
}

template <typename E, int ROLE>
__global__ void __launch_bounds__(kThreads) k_spmv_bsr3_rows(MatDev A, SolveState* st) {
    typedef E C;
    constexpr int NACC = RoleAcc<ROLE>::value;
    if (ROLE != ROLE_GEN && st->res.done) return;
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    bsr3_rows_body<E, ROLE>(A, x, y, u, acc, blockIdx.x, gridDim.x);
    write_partials<NACC>(st, acc);
}

}  // namespace msolve

namespace msolve {

// ------------------------------------------------------------------------------------------
// PTX wrappers: mbarrier + 1-D bulk async copy (TMA engine, SASS UBLKCP) + L2 cache policies.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
// global -> shared bulk copy; bytes % 16 == 0, both addresses 16-byte aligned; completes on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}
// x gathers of the BSR3 kernel: plain read-only loads (hinted 16-byte loads are slower on B200, profiles/r01_sweeps.md)
template <typename C> __device__ __forceinline__ C ld_hint(const C* p, uint64_t) { return __ldg(p); }

// ------------------------------------------------------------------------------------------
// BSR3, TMA-staged (the SU(3) lattice kernel).  Persistent CTAs, CPS of them per SM.  A producer
// thread streams tiles of TB block rows -- the tile's 3x3 blocks and its block-column indices
// are one contiguous byte range each -- into a STAGES-deep shared-memory ring with 1-D bulk
// async copies (evict-first in L2: the matrix is read once per SpMV), signalled by mbarriers.
// Phase 1: one consumer thread per 3x3 BLOCK gathers its x 3-vector ONCE (through L1/L2: every
// x element is used by its 2d+1 neighbour rows; a software pipeline issues the gathers of the
// next tile before the current one is multiplied), multiplies the block out of shared
// memory and leaves a 3-vector partial in shared memory; all gathers of a tile are in flight
// at once.  Phase 2 (after one named barrier): one thread per scalar row sums its row's
// partials, writes y and feeds the fused dot products.
// Tile table (A.aux, built at create time): int4 {row_begin, row_end, block_begin, block_end},
// block_begin % 4 == 0 so that every bulk copy is 16-byte aligned for both dtypes.
// ------------------------------------------------------------------------------------------
template <typename E, int TB> struct BsrTmaCfg {
    static constexpr int kMaxBlocks = 9 * TB;
    static constexpr int kConsumers = (kMaxBlocks + 31) / 32 * 32;
    static constexpr int kThreadsTotal = kConsumers + 32;
    static constexpr int kValBytes = kMaxBlocks * 9 * (int)sizeof(E);
    static constexpr int kIdxBytes = kMaxBlocks * 4;
    static constexpr int kStageBytes = kValBytes + kIdxBytes;
    static constexpr int kPartBytes = kMaxBlocks * 3 * (int)sizeof(E);       // one partial buffer
    static constexpr int smem_bytes(int stages) { return stages * kStageBytes + 2 * kPartBytes + 2 * stages * 8; }
};

template <typename E, int TB, int STAGES, int CPS, int ROLE>
__global__ void __launch_bounds__(BsrTmaCfg<E, TB>::kThreadsTotal, CPS) k_spmv_bsr3_tma(MatDev A, SolveState* st) {
    typedef E C;
    typedef BsrTmaCfg<E, TB> Cfg;
    constexpr int NACC = RoleAcc<ROLE>::value;
    constexpr int NCT = Cfg::kConsumers;
    constexpr int NCW = NCT / 32;
    if (ROLE != ROLE_GEN && st->res.done) return;
    extern __shared__ __align__(128) unsigned char smem[];
    C* part = (C*)(smem + STAGES * Cfg::kStageBytes);
    uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::kStageBytes + 2 * Cfg::kPartBytes);
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, NCW); }
        mbar_fence_init();
    }
    __syncthreads();
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    const int4* __restrict__ tiles = (const int4*)A.aux;
    const int ntiles = A.aux_count;
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    int stage = 0;
    uint32_t phase = 0;
    if (threadIdx.x >= NCT) {
        // ---------------- producer: one elected lane of the last warp
        if (threadIdx.x == NCT) {
            // the matrix is read once per SpMV: evict-first, unless it is small enough to stay in L2 between SpMVs
            const uint64_t pol = policy_matrix(A.mat_keep);
            const C* __restrict__ val = (const C*)A.val;
            int t = blockIdx.x;
            int4 e = t < ntiles ? tiles[t] : make_int4(0, 0, 0, 0);
            while (t < ntiles) {
                const int tn = t + gridDim.x;
                const int4 en = tn < ntiles ? tiles[tn] : make_int4(0, 0, 0, 0);
                mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                unsigned char* sb = smem + stage * Cfg::kStageBytes;
                const uint32_t nb = (uint32_t)(e.w - e.z);
                const uint32_t vbytes = nb * 9u * (uint32_t)sizeof(C), ibytes = nb * 4u;
                const uint32_t vb16 = vbytes & ~15u, ib16 = ibytes & ~15u;
                const unsigned char* vsrc = (const unsigned char*)(val + (long long)e.z * 9);
                const unsigned char* isrc = (const unsigned char*)(A.colidx + e.z);
                // ragged tail of the very last tile: < 16 bytes each, copied through the generic proxy
                for (uint32_t o = vb16; o < vbytes; o += 4) *(uint32_t*)(sb + o) = *(const uint32_t*)(vsrc + o);
                for (uint32_t o = ib16; o < ibytes; o += 4) *(uint32_t*)(sb + Cfg::kValBytes + o) = *(const uint32_t*)(isrc + o);
                mbar_expect_tx(full0 + 8 * stage, vb16 + ib16);
                if (vb16) bulk_g2s(smem_u32(sb), vsrc, vb16, full0 + 8 * stage, pol);
                if (ib16) bulk_g2s(smem_u32(sb + Cfg::kValBytes), isrc, ib16, full0 + 8 * stage, pol);
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                t = tn; e = en;
            }
        }
    } else {
        // ---------------- consumers.  Software-pipelined: the x gathers of tile t+1 are issued
        // (into registers) before tile t is multiplied, so their L2 latency overlaps the math,
        // the named barrier and phase 2 of tile t.  Tile-table entries are fetched two ahead.
        const uint64_t polx = policy_evict_last();
        const int tid = threadIdx.x;
        const int lbr = tid / 3, rr = tid - 3 * lbr;     // phase-2 role: scalar row (lbr, rr)
        const int32_t* __restrict__ browptr = A.rowptr;
        const int G = gridDim.x;
        int pbuf = 0;
        int t = blockIdx.x;
        const int4 zero4 = make_int4(0, 0, 0, 0);
        int4 e = t < ntiles ? tiles[t] : zero4;
        int4 en = t + G < ntiles ? tiles[t + G] : zero4;
        C xn0 = cmake<C>(0.0, 0.0), xn1 = xn0, xn2 = xn0;
        if (t < ntiles) {
            mbar_wait(full0, 0u);
            if (tid < e.w - e.z) {
                const int32_t c = ((const int32_t*)(smem + Cfg::kValBytes))[tid];
                const C* xv = x + 3ll * c;
                xn0 = ld_hint(xv, polx); xn1 = ld_hint(xv + 1, polx); xn2 = ld_hint(xv + 2, polx);
            }
        }
        while (t < ntiles) {
            const int tn = t + G;
            const int4 enn = tn + G < ntiles ? tiles[tn + G] : zero4;
            const int nb = e.w - e.z;
            const bool rvalid = lbr < e.y - e.x;
            int jb = 0, je = 0;
            if (rvalid) { jb = browptr[e.x + lbr] - e.z; je = browptr[e.x + lbr + 1] - e.z; }
            const C x0 = xn0, x1 = xn1, x2 = xn2;
            int nstage = stage + 1;
            uint32_t nphase = phase;
            if (nstage == STAGES) { nstage = 0; nphase ^= 1u; }
            if (tn < ntiles) {                                // gathers of the NEXT tile
                mbar_wait(full0 + 8 * nstage, nphase);
                if (tid < en.w - en.z) {
                    const int32_t c = ((const int32_t*)(smem + nstage * Cfg::kStageBytes + Cfg::kValBytes))[tid];
                    const C* xv = x + 3ll * c;
                    xn0 = ld_hint(xv, polx); xn1 = ld_hint(xv + 1, polx); xn2 = ld_hint(xv + 2, polx);
                }
            }
            C* pb = part + pbuf * (Cfg::kMaxBlocks * 3);
            if (tid < nb) {                                   // phase 1: block `tid` of the tile
                const C* blk = (const C*)(smem + stage * Cfg::kStageBytes) + tid * 9;
                C a[9];
#pragma unroll
                for (int k = 0; k < 9; ++k) a[k] = blk[k];
#pragma unroll
                for (int r3 = 0; r3 < 3; ++r3) {
                    C v = cmul(a[3 * r3], x0);
                    v = cfma(a[3 * r3 + 1], x1, v);
                    v = cfma(a[3 * r3 + 2], x2, v);
                    pb[tid * 3 + r3] = v;
                }
            }
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * stage);     // this warp no longer reads the stage
            asm volatile("bar.sync 1, %0;" ::"n"(NCT) : "memory");     // partials visible to all consumers
            if (rvalid) {                                     // phase 2: scalar row (lbr, rr)
                C sum = cmake<C>(0.0, 0.0);
                for (int j = jb; j < je; ++j) sum = cadd(sum, pb[j * 3 + rr]);
                const long long row = 3ll * (e.x + lbr) + rr;
                y[row] = sum;
                role_epilogue<C, ROLE>(acc, row, sum, x, u);
            }
            pbuf ^= 1;
            stage = nstage; phase = nphase;
            t = tn; e = en; en = enn;
        }
    }
    write_partials<NACC>(st, acc);
}

}  // namespace msolve
