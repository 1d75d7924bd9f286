// spmv_merge.cuh -- merge-path CSR SpMV for irregular rows (the
// "merge-path CSR" variant; Alg. 1 l.18-19; BASELINE config 5: row lengths
// power-law in [5,200]).
//
// The merge path is the monotone staircase through the (row-end, non-zero) grid: consuming item
// (i,k) either ends row i (when k == rowptr[i+1]) or multiplies non-zero k.  The n + nnz items
// are cut into tiles of equal length at create time (host-side diagonal search, `MergeTiles` in
// msolve.cu), so every tile carries the same amount of work whatever the row lengths are: a
// tile may begin and end in the middle of a row.
//
// Per tile (persistent CTAs, CPS per SM, grid-stride over tiles):
//   * a producer thread streams the tile's values, column indices and row offsets -- three
//     contiguous, 16-byte-aligned byte ranges (tile boundaries sit at non-zero indices that are
//     multiples of 4) -- into a STAGES-deep shared-memory ring with 1-D bulk async copies (TMA
//     engine, SASS UBLKCP), evict-first in L2 (the matrix is read once per SpMV);
//   * phase 1: consumer thread j multiplies non-zero j by its gathered x value, in place in
//     shared memory (coalesced, conflict-free).  The gathers of tile t+1 are issued before tile
//     t is processed (software pipeline), so their L2 latency is hidden;
//   * phase 2: groups of g lanes (g = largest power of two with rows*g <= consumers) sum the
//     products of one row each; complete rows are written to y and feed the fused dots; the
//     partial sums of the (at most two) rows cut by the tile boundary go to a carry array.
// A small fix-up kernel then adds the carries of rows that span tiles in tile order, writes
// those rows and their share of the dots.  All sums have a fixed order: results are
// bit-reproducible for a given tile size.
#pragma once

#include "spmv.cuh"

namespace msolve {

template <typename E, int CAP> struct MergeCfg {
    typedef E C;
    static constexpr int kConsumers = 256;
    static constexpr int kThreadsTotal = kConsumers + 32;
    static constexpr int kDiag = CAP - 4;                 // merge items per tile (before 4-alignment of k)
    static constexpr int kIpt = CAP / kConsumers;         // non-zeros per consumer thread
    static constexpr int kRowCap = CAP + 8;               // row offsets staged per tile
    static constexpr int kValBytes = CAP * (int)sizeof(C);
    static constexpr int kIdxBytes = CAP * 4;
    static constexpr int kRowBytes = kRowCap * 4;
    static constexpr int kStageBytes = kValBytes + kIdxBytes + kRowBytes;
    static constexpr int smem_bytes(int stages) { return stages * kStageBytes + 2 * stages * 8; }
    static_assert(CAP % kConsumers == 0, "CAP must be a multiple of the consumer count");
};

// Per-CTA partials written behind those of a preceding kernel (the fix-up kernel appends).
template <int NACC>
__device__ __forceinline__ void write_partials_at(SolveState* st, double (&acc)[NACC], int offset, int total) {
    __shared__ double red2[NACC * 32];
    block_sum<NACC>(acc, red2);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int a = 0; a < NACC; ++a) st->partial[a * kMaxPartials + offset + blockIdx.x] = acc[a];
        if (blockIdx.x == 0) st->partial_count = total;
    }
}

template <typename E, int CAP, int STAGES, int CPS, int ROLE, bool PIN>
__global__ void __launch_bounds__(MergeCfg<E, CAP>::kThreadsTotal, CPS) k_spmv_csr_merge(MatDev A, SolveState* st) {
    typedef E C;
    typedef MergeCfg<E, CAP> Cfg;
    constexpr int NACC = RoleAcc<ROLE>::value;
    constexpr int NCT = Cfg::kConsumers;
    constexpr int NCW = NCT / 32;
    constexpr int IPT = Cfg::kIpt;
    if (ROLE != ROLE_GEN && st->res.done) return;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::kStageBytes);
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
    const int n = (int)A.n;
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
                const uint32_t nz = (uint32_t)(e.w - e.z);
                const uint32_t vbytes = nz * (uint32_t)sizeof(C), ibytes = nz * 4u;
                // row offsets rowptr[first .. last], first = i0 rounded down to a multiple of 4
                const int first = e.x & ~3;
                const int last = min(e.y + 1, n);
                int cnt = min(last - first + 1, Cfg::kRowCap);
                if (first + ((cnt + 3) & ~3) <= n + 1) cnt = (cnt + 3) & ~3;      // over-read inside the array
                const uint32_t rbytes = (uint32_t)cnt * 4u;
                const uint32_t vb16 = vbytes & ~15u, ib16 = ibytes & ~15u, rb16 = rbytes & ~15u;
                const unsigned char* vsrc = (const unsigned char*)(val + e.z);
                const unsigned char* isrc = (const unsigned char*)(A.colidx + e.z);
                const unsigned char* rsrc = (const unsigned char*)(A.rowptr + first);
                unsigned char* vdst = sb;
                unsigned char* idst = sb + Cfg::kValBytes;
                unsigned char* rdst = sb + Cfg::kValBytes + Cfg::kIdxBytes;
                // ragged tails (< 16 bytes, only at the very end of the arrays): generic proxy
                for (uint32_t o = vb16; o < vbytes; o += 4) *(uint32_t*)(vdst + o) = *(const uint32_t*)(vsrc + o);
                for (uint32_t o = ib16; o < ibytes; o += 4) *(uint32_t*)(idst + o) = *(const uint32_t*)(isrc + o);
                for (uint32_t o = rb16; o < rbytes; o += 4) *(uint32_t*)(rdst + o) = *(const uint32_t*)(rsrc + o);
                mbar_expect_tx(full0 + 8 * stage, vb16 + ib16 + rb16);
                if (vb16) bulk_g2s(smem_u32(vdst), vsrc, vb16, full0 + 8 * stage, pol);
                if (ib16) bulk_g2s(smem_u32(idst), isrc, ib16, full0 + 8 * stage, pol);
                if (rb16) bulk_g2s(smem_u32(rdst), rsrc, rb16, full0 + 8 * stage, pol);
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                t = tn; e = en;
            }
        }
    } else {
        // ---------------- consumers
        const int tid = threadIdx.x;
        const uint64_t polx = policy_evict_last();
        const int32_t* __restrict__ rowptr = A.rowptr;
        C* head = (C*)A.carry;
        C* tail = head + ntiles;
        const int G = gridDim.x;
        int t = blockIdx.x;
        const int4 zero4 = make_int4(0, 0, 0, 0);
        int4 e = t < ntiles ? tiles[t] : zero4;
        int4 en = t + G < ntiles ? tiles[t + G] : zero4;
        C xn[IPT];
#pragma unroll
        for (int i = 0; i < IPT; ++i) xn[i] = cmake<C>(0.0, 0.0);
        if (t < ntiles) {
            mbar_wait(full0, 0u);
            const int32_t* cols = (const int32_t*)(smem + Cfg::kValBytes);
            const int nz = e.w - e.z;
#pragma unroll
            for (int i = 0; i < IPT; ++i) {
                const int j = tid + i * NCT;
                if (j < nz) xn[i] = ld_xg<PIN>(x + cols[j], polx);
            }
        }
        while (t < ntiles) {
            const int tn = t + G;
            const int4 enn = tn + G < ntiles ? tiles[tn + G] : zero4;
            C xc[IPT];
#pragma unroll
            for (int i = 0; i < IPT; ++i) xc[i] = xn[i];
            int nstage = stage + 1;
            uint32_t nphase = phase;
            if (nstage == STAGES) { nstage = 0; nphase ^= 1u; }
            if (tn < ntiles) {                                   // gathers of the NEXT tile
                mbar_wait(full0 + 8 * nstage, nphase);
                const int32_t* cols = (const int32_t*)(smem + nstage * Cfg::kStageBytes + Cfg::kValBytes);
                const int nzn = en.w - en.z;
#pragma unroll
                for (int i = 0; i < IPT; ++i) {
                    const int j = tid + i * NCT;
                    if (j < nzn) xn[i] = ld_xg<PIN>(x + cols[j], polx);
                }
            }
            // phase 1: products, in place
            unsigned char* sb = smem + stage * Cfg::kStageBytes;
            C* vals = (C*)sb;
            const int32_t* rps = (const int32_t*)(sb + Cfg::kValBytes + Cfg::kIdxBytes);
            const int k0 = e.z, k1 = e.w, nz = k1 - k0;
#pragma unroll
            for (int i = 0; i < IPT; ++i) {
                const int j = tid + i * NCT;
                if (j < nz) vals[j] = cmul(vals[j], xc[i]);
            }
            asm volatile("bar.sync 1, %0;" ::"n"(NCT) : "memory");
            // phase 2: one group of g lanes per row
            const int rbase = e.x & ~3;
            const int R = e.y - e.x + (e.y < n ? 1 : 0);          // rows i0 .. min(i1, n-1)
            int g = 32, lg = 5;
            while (g > 1 && R * g > NCT) { g >>= 1; --lg; }
            const int NG = NCT >> lg;
            const int gid = tid >> lg, l = tid & (g - 1);
            for (int base = 0; base < R; base += NG) {
                const int rr = base + gid;
                const int r = e.x + rr;
                const bool valid = rr < R;
                int rs = 0, re = 0;
                if (valid) {
                    const int o = r - rbase;
                    rs = o < Cfg::kRowCap ? rps[o] : rowptr[r];
                    re = o + 1 < Cfg::kRowCap ? rps[o + 1] : rowptr[r + 1];
                }
                const bool started = rs >= k0, ends = r < e.y;
                const int lo = max(rs, k0) - k0, hi = min(re, k1) - k0;
                C sum = cmake<C>(0.0, 0.0);
                if (valid) {
                    for (int j = lo + l; j < hi; j += g) sum = cadd(sum, vals[j]);
                }
                for (int o = g >> 1; o > 0; o >>= 1) sum = cshfl_xor_add(sum, o);
                if (valid && l == 0) {
                    if (started && ends) {
                        y[r] = sum;
                        role_epilogue<C, ROLE>(acc, r, sum, x, u);
                    } else if (!started) {
                        head[t] = sum;                            // row i0 began in an earlier tile
                    } else if (hi > lo) {
                        tail[t] = sum;                            // row i1 continues in the next tile
                    }
                }
            }
            // the stage was written through the generic proxy (products): order those writes
            // before the async-proxy refill, then hand the stage back
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * stage);
            stage = nstage; phase = nphase;
            t = tn; e = en; en = enn;
        }
    }
    write_partials_at<NACC>(st, acc, 0, gridDim.x);
}

// Rows cut by tile boundaries: y[row] = tail of the tile the row begins in + the heads of the
// following tiles up to the one the row ends in, summed in tile order by one thread.
template <typename E, int ROLE>
__global__ void __launch_bounds__(kThreads) k_spmv_csr_merge_fixup(MatDev A, SolveState* st, int main_grid) {
    typedef E C;
    constexpr int NACC = RoleAcc<ROLE>::value;
    if (ROLE != ROLE_GEN && st->res.done) return;
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    const int4* __restrict__ tiles = (const int4*)A.aux;
    const int ntiles = A.aux_count;
    const int n = (int)A.n;
    const C* head = (const C*)A.carry;
    const C* tail = head + ntiles;
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    const int stride = gridDim.x * blockDim.x;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < ntiles; t += stride) {
        const int4 e = tiles[t];
        if (e.y >= n) continue;
        const int rs = A.rowptr[e.y];
        if (rs < e.z || e.w <= rs) continue;                      // no row begins here and continues
        C sum = tail[t];
        for (int t2 = t + 1; t2 < ntiles; ++t2) {
            const int4 f = tiles[t2];
            sum = cadd(sum, head[t2]);
            if (f.x < f.y) break;                                 // the row ends in tile t2
        }
        y[e.y] = sum;
        role_epilogue<C, ROLE>(acc, e.y, sum, x, u);
    }
    write_partials_at<NACC>(st, acc, main_grid, main_grid + gridDim.x);
}

}  // namespace msolve
