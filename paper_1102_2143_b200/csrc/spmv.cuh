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

enum { ROLE_CG = 0, ROLE_B1 = 1, ROLE_B2 = 2, ROLE_GEN = 3 };

template <int ROLE> struct RoleAcc { static constexpr int value = ROLE == ROLE_CG ? 1 : (ROLE == ROLE_B2 ? 5 : 2); };

template <typename C, int ROLE>
__device__ __forceinline__ void role_vectors(const SolveState* st, const C*& x, C*& y, const C*& u) {
    if (ROLE == ROLE_CG)  { x = (const C*)st->h.p; y = (C*)st->h.q; u = nullptr; }
    if (ROLE == ROLE_B1)  { x = (const C*)st->h.p; y = (C*)st->h.q; u = (const C*)st->h.b; }
    if (ROLE == ROLE_B2)  { x = (const C*)st->h.s; y = (C*)st->h.t; u = (const C*)st->h.b; }
    if (ROLE == ROLE_GEN) { x = (const C*)st->h.sp_x; y = (C*)st->h.sp_y; u = (const C*)st->h.sp_u; }
}

// Fused reductions for one finished row (all accumulation in fp64, R14).
template <typename C, int ROLE>
__device__ __forceinline__ void role_epilogue(double* acc, long long row, C yi, const C* x, const C* u) {
    const double yr = yi.x, ym = yi.y;
    if (ROLE == ROLE_CG) {
        const C xi = x[row];
        acc[0] += (double)xi.x * yr + (double)xi.y * ym;
    } else if (ROLE == ROLE_B1 || ROLE == ROLE_GEN) {
        const C ui = u[row];
        acc[0] += (double)ui.x * yr + (double)ui.y * ym;       // conj(u) y
        acc[1] += (double)ui.x * ym - (double)ui.y * yr;
    } else {
        const C xi = x[row];
        const C ui = u[row];
        acc[0] += yr * (double)xi.x + ym * (double)xi.y;        // conj(y) x  = <t,s>
        acc[1] += yr * (double)xi.y - ym * (double)xi.x;
        acc[2] += yr * yr + ym * ym;                            // <t,t>
        acc[3] += (double)ui.x * yr + (double)ui.y * ym;        // <r0,t>
        acc[4] += (double)ui.x * ym - (double)ui.y * yr;
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
template <typename T, int LANES, int ROLE>
__global__ void __launch_bounds__(kThreads) k_spmv_csr_vector(MatDev A, SolveState* st) {
    typedef typename Cx<T>::type C;
    constexpr int NACC = RoleAcc<ROLE>::value;
    if (ROLE != ROLE_GEN && st->res.done) return;
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    const C* __restrict__ val = (const C*)A.val;
    const int32_t* __restrict__ colidx = A.colidx;
    const int32_t* __restrict__ rowptr = A.rowptr;
    constexpr int RPW = 32 / LANES;  // rows per warp
    const int lane = threadIdx.x & 31;
    const int sub = lane % LANES;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    for (long long base = warp * RPW; base < A.n; base += nwarps * RPW) {
        const long long row = base + lane / LANES;
        const bool valid = row < A.n;
        int j = 0, e = 0;
        if (valid) { j = rowptr[row] + sub; e = rowptr[row + 1]; }
        C sum = cmake<C>(0.0, 0.0);
#pragma unroll 4
        for (; j < e; j += LANES) {
            const int c = ld_stream(colidx + j);
            const C v = ld_stream(val + j);
            sum = cfma(v, ld_ro(x + c), sum);
        }
#pragma unroll
        for (int o = LANES / 2; o > 0; o >>= 1) {
            sum.x += __shfl_xor_sync(0xffffffffu, sum.x, o);
            sum.y += __shfl_xor_sync(0xffffffffu, sum.y, o);
        }
        if (valid && sub == 0) {
            y[row] = sum;
            role_epilogue<C, ROLE>(acc, row, sum, x, u);
        }
    }
    write_partials<NACC>(st, acc);
}

// ------------------------------------------------------------------------------------------
// BSR3, one thread per scalar row (first, simple variant): thread (br, r) walks the blocks of
// block row br and multiplies row r of every 3x3 block with the 3-vector x[3*bcol .. +3].
// The three threads of a block row read one contiguous 144-byte (c128) block between them.
// ------------------------------------------------------------------------------------------
template <typename T, int ROLE>
__global__ void __launch_bounds__(kThreads) k_spmv_bsr3_rows(MatDev A, SolveState* st) {
    typedef typename Cx<T>::type C;
    constexpr int NACC = RoleAcc<ROLE>::value;
    if (ROLE != ROLE_GEN && st->res.done) return;
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    const C* __restrict__ val = (const C*)A.val;
    const int32_t* __restrict__ bcol = A.colidx;
    const int32_t* __restrict__ browptr = A.rowptr;
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long row = (long long)blockIdx.x * blockDim.x + threadIdx.x; row < A.n; row += stride) {
        const long long br = row / 3;
        const int rr = (int)(row - 3 * br);
        const int jb = browptr[br], je = browptr[br + 1];
        C sum = cmake<C>(0.0, 0.0);
#pragma unroll 3
        for (int j = jb; j < je; ++j) {
            const C* blk = val + (long long)j * 9 + rr * 3;
            const C* xv = x + 3ll * bcol[j];
            const C a0 = ld_stream(blk), a1 = ld_stream(blk + 1), a2 = ld_stream(blk + 2);
            sum = cfma(a0, ld_ro(xv), sum);
            sum = cfma(a1, ld_ro(xv + 1), sum);
            sum = cfma(a2, ld_ro(xv + 2), sum);
        }
        y[row] = sum;
        role_epilogue<C, ROLE>(acc, row, sum, x, u);
    }
    write_partials<NACC>(st, acc);
}

}  // namespace msolve
