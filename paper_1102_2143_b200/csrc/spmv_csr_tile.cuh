// spmv_csr_tile.cuh -- TMA-staged vector-CSR SpMV for short rows (the
// "vector-CSR for short regular lattice rows" variant with the matrix staged through shared
// memory by the TMA engine; Alg. 1 l.18-19; BASELINE config 4 as CSR: 27
// non-zeros per row).
//
// Same row mapping as k_spmv_csr_vector (LANES lanes per row, lane l of a row takes non-zeros
// l, l+LANES, ... and the row sum is a shuffle reduction), but the matrix does not go through
// the load/store units of the consumer warps:
//   * a tile is TR = 128 / LANES consecutive rows; its values and column indices are ONE
//     contiguous byte range each (widened to multiples of 4 non-zeros so that both ranges are
//     16-byte aligned), streamed by a producer thread into a STAGES-deep shared-memory ring
//     with 1-D bulk async copies (SASS UBLKCP), evict-first in L2 -- the matrix is read once
//     per SpMV and must not displace x, which every row's 2d+1 neighbours re-read from L2;
//   * consumers are warp-autonomous (no CTA barrier): a warp waits for the stage, issues the x
//     gathers of tile t+1 (column indices out of shared memory) before it multiplies tile t,
//     accumulates in registers and hands the stage back through the `empty` mbarrier;
//   * row offsets of tile t+2 are prefetched from global memory while tile t is computed.
// Eligible when every row has at most LANES * U non-zeros (create-time check); tiles are fixed
// (tile t = rows [t*TR, (t+1)*TR)), so there is no tile table.
#pragma once

#include "spmv.cuh"

namespace msolve {

template <typename E, int LANES, int U> struct CsrTileCfg {
    static constexpr int kConsumers = 128;
    static constexpr int kThreadsTotal = kConsumers + 32;
    static constexpr int kRows = kConsumers / LANES;          // rows per tile
    static constexpr int kCap = kConsumers * U + 8;           // non-zeros staged per tile (+ alignment slack)
    static constexpr int kValBytes = kCap * (int)sizeof(E);
    static constexpr int kIdxBytes = kCap * 4;
    static constexpr int kStageBytes = kValBytes + kIdxBytes; // multiple of 16
    static constexpr int smem_bytes(int stages) { return stages * kStageBytes + 2 * stages * 8 + stages * 16; }
};

// x gather: elements of at most 8 bytes go through a hinted load (policy chosen at run time:
// evict_last when x fits in L2 beside the stream); 16-byte elements use the plain nc load
// (hinted 16-byte loads are slower on B200, profiles/r01_sweeps.md).
template <typename E> __device__ __forceinline__ E ld_xt(const E* p, uint64_t pol) { return ld_xg<true>(p, pol); }
template <> __device__ __forceinline__ double2 ld_xt<double2>(const double2* p, uint64_t) { return __ldg(p); }

template <typename E, int LANES, int U, int STAGES, int CPS, int ROLE>
__global__ void __launch_bounds__(CsrTileCfg<E, LANES, U>::kThreadsTotal, CPS) k_spmv_csr_tile(MatDev A, SolveState* st) {
    typedef E C;
    typedef CsrTileCfg<E, LANES, U> Cfg;
    constexpr int NACC = RoleAcc<ROLE>::value;
    constexpr int NCT = Cfg::kConsumers;
    constexpr int NCW = NCT / 32;
    constexpr int TR = Cfg::kRows;
    if (ROLE != ROLE_GEN && st->res.done) return;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::kStageBytes);
    int* meta = (int*)(smem + STAGES * Cfg::kStageBytes + 2 * STAGES * 8);   // per stage: first staged non-zero
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, NCW); }
        mbar_fence_init();
    }
    __syncthreads();
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    const int32_t* __restrict__ rowptr = A.rowptr;
    const int n = (int)A.n;
    const int nnz = (int)A.nnz;
    const int ntiles = (n + TR - 1) / TR;
    const int G = gridDim.x;
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
            int ka = 0, kb = 0;
            if (t < ntiles) { ka = rowptr[t * TR]; kb = rowptr[min(n, (t + 1) * TR)]; }
            while (t < ntiles) {
                const int tn = t + G;
                int kan = 0, kbn = 0;
                if (tn < ntiles) { kan = rowptr[tn * TR]; kbn = rowptr[min(n, (tn + 1) * TR)]; }
                mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                unsigned char* sb = smem + stage * Cfg::kStageBytes;
                const int k0 = ka & ~3;
                const int k1 = min(nnz, (kb + 3) & ~3);
                const uint32_t nz = (uint32_t)(k1 - k0);
                const uint32_t vbytes = nz * (uint32_t)sizeof(C), ibytes = nz * 4u;
                const uint32_t vb16 = vbytes & ~15u, ib16 = ibytes & ~15u;
                const unsigned char* vsrc = (const unsigned char*)(val + k0);
                const unsigned char* isrc = (const unsigned char*)(A.colidx + k0);
                // ragged tail (< 16 bytes, only at the very end of the arrays): generic proxy
                for (uint32_t o = vb16; o < vbytes; o += 4) *(uint32_t*)(sb + o) = *(const uint32_t*)(vsrc + o);
                for (uint32_t o = ib16; o < ibytes; o += 4) *(uint32_t*)(sb + Cfg::kValBytes + o) = *(const uint32_t*)(isrc + o);
                meta[4 * stage] = k0;
                mbar_expect_tx(full0 + 8 * stage, vb16 + ib16);
                if (vb16) bulk_g2s(smem_u32(sb), vsrc, vb16, full0 + 8 * stage, pol);
                if (ib16) bulk_g2s(smem_u32(sb + Cfg::kValBytes), isrc, ib16, full0 + 8 * stage, pol);
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                t = tn; ka = kan; kb = kbn;
            }
        }
    } else {
        // ---------------- consumers: lane group (rl, l) owns row t*TR + rl of every tile
        const uint64_t polx = A.x_pin ? policy_evict_last() : policy_evict_normal();
        const int tid = threadIdx.x;
        const int rl = tid / LANES, l = tid % LANES;
        int t = blockIdx.x;
        // row offsets of the current, next and next-but-one tile
        int rs = 0, re = 0, rsn = 0, ren = 0;
        if (t < ntiles && t * TR + rl < n) { rs = rowptr[t * TR + rl]; re = rowptr[t * TR + rl + 1]; }
        if (t + G < ntiles && (t + G) * TR + rl < n) { rsn = rowptr[(t + G) * TR + rl]; ren = rowptr[(t + G) * TR + rl + 1]; }
        C xn[U];
#pragma unroll
        for (int i = 0; i < U; ++i) xn[i] = cmake<C>(0.0, 0.0);
        if (t < ntiles) {
            mbar_wait(full0, 0u);
            const int32_t* cols = (const int32_t*)(smem + Cfg::kValBytes);
            const int k0 = meta[0];
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const int j = rs + l + i * LANES;
                if (j < re) xn[i] = ld_xt<C>(x + cols[j - k0], polx);
            }
        }
        while (t < ntiles) {
            const int tn = t + G, tnn = tn + G;
            int rsnn = 0, renn = 0;
            if (tnn < ntiles && tnn * TR + rl < n) { rsnn = rowptr[tnn * TR + rl]; renn = rowptr[tnn * TR + rl + 1]; }
            C xc[U];
#pragma unroll
            for (int i = 0; i < U; ++i) xc[i] = xn[i];
            int nstage = stage + 1;
            uint32_t nphase = phase;
            if (nstage == STAGES) { nstage = 0; nphase ^= 1u; }
            if (tn < ntiles) {                                   // gathers of the NEXT tile
                mbar_wait(full0 + 8 * nstage, nphase);
                const int32_t* cols = (const int32_t*)(smem + nstage * Cfg::kStageBytes + Cfg::kValBytes);
                const int k0n = meta[4 * nstage];
#pragma unroll
                for (int i = 0; i < U; ++i) {
                    const int j = rsn + l + i * LANES;
                    if (j < ren) xn[i] = ld_xt<C>(x + cols[j - k0n], polx);
                }
            }
            const C* vals = (const C*)(smem + stage * Cfg::kStageBytes);
            const int k0 = meta[4 * stage];
            C sum = cmake<C>(0.0, 0.0);
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const int j = rs + l + i * LANES;
                if (j < re) sum = cfma(vals[j - k0], xc[i], sum);
            }
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * stage);     // this warp no longer reads the stage
#pragma unroll
            for (int o = LANES / 2; o > 0; o >>= 1) sum = cshfl_xor_add(sum, o);
            const int row = t * TR + rl;
            if (l == 0 && row < n) {
                y[row] = sum;
                role_epilogue<C, ROLE>(acc, row, sum, x, u);
            }
            stage = nstage; phase = nphase;
            t = tn; rs = rsn; re = ren; rsn = rsnn; ren = renn;
        }
    }
    write_partials<NACC>(st, acc);
}

}  // namespace msolve
