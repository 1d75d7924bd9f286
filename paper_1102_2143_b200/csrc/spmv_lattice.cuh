// spmv_lattice.cuh -- matrix-free gauged lattice operator with SU(3) links (the
// "custom linear operator" hook the paper advertises, applied to the operator of
// BASELINE configs 2-4):
//
//   (A x)(s) = D x(s) - sum_mu [ c_f U_mu(s) x(s+mu) + c_b U_mu(s-mu)^dagger x(s-mu) ]
//
// read straight from the link field links[mu][s] = U_mu(s) (3x3 complex, row-major) instead of an
// assembled BSR3 matrix: 4 x 144 B of links per site (c128) instead of 9 x 148 B of blocks and
// indices.  Every link is used twice (forward at s, backward at s+mu); the second use is an L2 hit.
//
// Site index s = x0 + L0 (x1 + L1 (x2 + L2 x3)), periodic; scalar row = 3 s + colour.
//
// k_spmv_lat_tma: a tile is T consecutive x0-rows (T L0 <= NS sites, contiguous in memory).  All
// operands of a tile are contiguous byte ranges, so the producer thread moves EVERYTHING with 1-D
// bulk async copies (TMA engine) into a shared-memory ring -- there is not a single gather:
//   * forward links U_mu(s) of the tile's sites: one range per direction;
//   * backward links U_mu(s-mu), mu >= 1: per x0-row one range (the row at coordinate x_mu - 1);
//     mu = 0: U_0(s-0) is the forward link of the left neighbour in the same row, already staged;
//   * x of the tile's sites (one range), and per x0-row the 2(d-1) neighbour rows; the mu = 0
//     neighbours are the same row rotated by one site.
// Phase 1: one consumer thread per (direction term, site) multiplies its 3x3 link (or its conjugate
// transpose) with the neighbour's 3-vector out of shared memory and leaves a 3-vector partial.
// Phase 2 (one named barrier later): one thread per scalar row combines the 2d partials with the
// diagonal term, writes y (coalesced) and feeds the fused dot products.
#pragma once

#include "spmv.cuh"

namespace msolve {

// acc + conj(a) * b
template <typename C> __device__ __forceinline__ C cfma_conj(C a, C b, C acc) {
    acc.x += a.x * b.x; acc.x += a.y * b.y;
    acc.y += a.x * b.y; acc.y -= a.y * b.x;
    return acc;
}

// y = D xi - (cf f + cb g)
template <typename C, typename T>
__device__ __forceinline__ C lat_combine(T dg, C xi, T cf, C f, T cb, C g) {
    C r;
    r.x = dg * xi.x - (cf * f.x + cb * g.x);
    r.y = dg * xi.y - (cf * f.y + cb * g.y);
    return r;
}

// ------------------------------------------------------------------------------------------
// Fallback (any extents): one thread per scalar row, operands through L1/L2.
// ------------------------------------------------------------------------------------------
template <typename E, int ROLE, bool NC = true>
__device__ __forceinline__ void lat_rows_body(const MatDev& A, const E* x, E* y, const E* u, double* acc, int cta, int ncta) {
    typedef E C;
    typedef typename RealOf<E>::type T;
    const C* __restrict__ links = (const C*)A.val;
    const long long vol = A.lat_vol;
    const int nd = A.lat_ndim;
    const T dg = (T)A.lat_diag, cf = (T)A.lat_cf, cb = (T)A.lat_cb;
    const long long stride = (long long)ncta * blockDim.x;
    for (long long row = (long long)cta * blockDim.x + threadIdx.x; row < A.n; row += stride) {
        const long long s = row / 3;
        const int r = (int)(row - 3 * s);
        C f = cmake<C>(0.0, 0.0), g = f;
        long long rem = s, str = 1;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            if (mu >= nd) break;
            const int L = A.lat_ext[mu];
            const int c = (int)(rem % L);
            rem /= L;
            const long long sf = s + (c + 1 == L ? -(long long)(L - 1) * str : str);
            const long long sb = s + (c == 0 ? (long long)(L - 1) * str : -str);
            const C* U = links + ((long long)mu * vol + s) * 9 + 3 * r;      // row r of U_mu(s)
            const C* xf = x + 3 * sf;
            f = cfma(ld_ro(U), NC ? ld_ro(xf) : xf[0], f);
            f = cfma(ld_ro(U + 1), NC ? ld_ro(xf + 1) : xf[1], f);
            f = cfma(ld_ro(U + 2), NC ? ld_ro(xf + 2) : xf[2], f);
            const C* V = links + ((long long)mu * vol + sb) * 9 + r;         // column r of U_mu(s-mu)
            const C* xb = x + 3 * sb;
            g = cfma_conj(ld_ro(V), NC ? ld_ro(xb) : xb[0], g);
            g = cfma_conj(ld_ro(V + 3), NC ? ld_ro(xb + 1) : xb[1], g);
            g = cfma_conj(ld_ro(V + 6), NC ? ld_ro(xb + 2) : xb[2], g);
            str *= L;
        }
        const C sum = lat_combine(dg, NC ? ld_ro(x + row) : x[row], cf, f, cb, g);
        y[row] = sum;
        role_epilogue<C, ROLE>(acc, row, sum, x, u);
    }
}

template <typename E, int ROLE>
__global__ void __launch_bounds__(kThreads) k_spmv_lat_rows(MatDev A, SolveState* st) {
    typedef E C;
    constexpr int NACC = RoleAcc<ROLE>::value;
    if (ROLE != ROLE_GEN && st->res.done) return;
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    lat_rows_body<E, ROLE>(A, x, y, u, acc, blockIdx.x, gridDim.x);
    write_partials<NACC>(st, acc);
}

// fused reductions with x_i and u_i already in registers (same sums as role_epilogue)
template <typename C, int ROLE>
__device__ __forceinline__ void lat_epilogue(double* acc, C yi, C xi, C ui) {
    if (ROLE == ROLE_CG) {
        acc[0] += cdot_re(xi, yi);
    } else if (ROLE == ROLE_B1 || ROLE == ROLE_GEN) {
        acc[0] += cdot_re(ui, yi);
        acc[1] += cdot_im(ui, yi);
    } else {
        acc[0] += cdot_re(yi, xi);
        acc[1] += cdot_im(yi, xi);
        acc[2] += cnorm2(yi);
        acc[3] += cdot_re(ui, yi);
        acc[4] += cdot_im(ui, yi);
    }
}

// Producer side of both tile kernels, run by ONE elected thread: waits for the stage, posts the byte
// count and issues the tile's bulk copies (d + 1 + 3 (d-1) per x0-row: 14 for one 4-D row).  Issuing
// is the bottleneck of these kernels (~0.1 us per copy and thread; spreading the copies over the
// lanes of a warp is slower still: UBLKCP is a uniform-datapath instruction), hence 32-bit coordinate
// arithmetic here and several producer warps in k_spmv_lat_warp.
// lattice geometry the producers need, read once per kernel into registers (the 64-bit division vol / L0 must not
// end up inside the issue loop: measured +8 % on the complex64 kernel when the compiler left it there)
struct LatGeom {
    int nd, L0, TR, nrows;
    unsigned ext1, ext2, ext3;
    long long vol;
};
__device__ __forceinline__ LatGeom lat_geom(const MatDev& A) {
    LatGeom g;
    g.nd = A.lat_ndim; g.L0 = A.lat_ext[0]; g.TR = A.lat_rows_per_tile;
    g.ext1 = (unsigned)A.lat_ext[1]; g.ext2 = (unsigned)A.lat_ext[2]; g.ext3 = (unsigned)A.lat_ext[3];
    g.vol = A.lat_vol;
    g.nrows = (int)(A.lat_vol / A.lat_ext[0]);
    return g;
}

template <typename C, int LINK_SLOT, int X_SLOT, int X_BASE>
__device__ __forceinline__ void lat_issue_tile(const LatGeom& G, const C* __restrict__ links, const C* x, unsigned char* sb,
                                               uint32_t bar, uint32_t empty_bar, uint32_t empty_parity, int t, uint64_t pol) {
    constexpr int SZ = (int)sizeof(C);
    const int nd = G.nd, L0 = G.L0, TR = G.TR;
    const long long vol = G.vol;
    const int nrows = G.nrows;
    const int row0 = t * TR;
    const int nr = min(TR, nrows - row0);
    const long long site0 = (long long)row0 * L0;
    const uint32_t ns = (uint32_t)(nr * L0);
    const uint32_t lrow = (uint32_t)(L0 * 9 * SZ), xrow = (uint32_t)(L0 * 3 * SZ);
    mbar_wait(empty_bar, empty_parity);
    mbar_expect_tx(bar, ns * (uint32_t)SZ * (uint32_t)(9 * nd + 3 + (nd - 1) * 15));
    for (int mu = 0; mu < nd; ++mu)                                     // forward links of the tile
        bulk_g2s(smem_u32(sb + mu * LINK_SLOT), links + ((long long)mu * vol + site0) * 9, ns * 9u * SZ, bar, pol);
    bulk_g2s(smem_u32(sb + X_BASE), x + 3 * site0, ns * 3u * SZ, bar, pol);
    for (int rt = 0; rt < nr; ++rt) {
        const unsigned row = (unsigned)(row0 + rt);                     // = x1 + L1 (x2 + L2 x3)
        unsigned rem = row, rs = 1;
#pragma unroll
        for (int mu = 1; mu < 4; ++mu) {
            if (mu >= nd) break;
            const unsigned L = mu == 1 ? G.ext1 : mu == 2 ? G.ext2 : G.ext3;
            const unsigned cm = rem % L;
            rem /= L;
            const long long rf = (long long)row + (cm + 1 == L ? -(long long)((L - 1) * rs) : (long long)rs);
            const long long rb = (long long)row + (cm == 0 ? (long long)((L - 1) * rs) : -(long long)rs);
            bulk_g2s(smem_u32(sb + (3 + mu) * LINK_SLOT + rt * lrow), links + ((long long)mu * vol + rb * L0) * 9, lrow, bar, pol);
            bulk_g2s(smem_u32(sb + X_BASE + mu * X_SLOT + rt * xrow), x + 3 * rf * L0, xrow, bar, pol);
            bulk_g2s(smem_u32(sb + X_BASE + (3 + mu) * X_SLOT + rt * xrow), x + 3 * rb * L0, xrow, bar, pol);
            rs *= L;
        }
    }
}

// ------------------------------------------------------------------------------------------
// TMA-staged tile kernel.
// ------------------------------------------------------------------------------------------
template <typename E, int NS> struct LatCfg {
    static constexpr int kConsumers = 8 * NS;                           // (term, site) pairs, d <= 4
    static constexpr int kThreadsTotal = kConsumers + 32;
    static constexpr int kLinkSlot = NS * 9 * (int)sizeof(E);           // one direction's links
    static constexpr int kXSlot = NS * 3 * (int)sizeof(E);              // one neighbour's x
    static constexpr int kXBase = 7 * kLinkSlot;                        // x slots behind the link slots
    static constexpr int kStageBytes = 7 * (kLinkSlot + kXSlot);
    static constexpr int kPartBytes = 9 * NS * 3 * (int)sizeof(E);      // 8 terms + a copy of x(s)
    static constexpr int smem_bytes(int stages) { return stages * kStageBytes + 2 * kPartBytes + 2 * stages * 8; }
    static_assert((NS & (NS - 1)) == 0, "NS must be a power of two");
};
// link slots: 0..3 = forward U_mu(s), mu = 0..3 ; 4..6 = backward U_mu(s-mu), mu = 1..3
// x slots   : 0 = x(s) ; 1..3 = x(s+mu), mu = 1..3 ; 4..6 = x(s-mu), mu = 1..3

template <typename E, int NS, int STAGES, int CPS, int ROLE>
__global__ void __launch_bounds__(LatCfg<E, NS>::kThreadsTotal, CPS) k_spmv_lat_tma(MatDev A, SolveState* st) {
    typedef E C;
    typedef typename RealOf<E>::type T;
    typedef LatCfg<E, NS> Cfg;
    constexpr int NACC = RoleAcc<ROLE>::value;
    constexpr int NCT = Cfg::kConsumers;
    constexpr int NCW = NCT / 32;
    constexpr int SZ = (int)sizeof(C);
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
    const int nd = A.lat_ndim;
    const int L0 = A.lat_ext[0];
    const int TR = A.lat_rows_per_tile;
    const long long vol = A.lat_vol;
    const long long nrows = vol / L0;                                    // x0-rows of the lattice
    const int ntiles = A.aux_count;
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    int stage = 0;
    uint32_t phase = 0;
    if (threadIdx.x >= NCT) {
        // ---------------- producer: one elected lane of the last warp
        if (threadIdx.x == NCT) {
            const C* __restrict__ links = (const C*)A.val;
            const uint64_t pol = policy_evict_normal();
            const LatGeom G = lat_geom(A);
            for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
                lat_issue_tile<C, Cfg::kLinkSlot, Cfg::kXSlot, Cfg::kXBase>(G, links, x, smem + stage * Cfg::kStageBytes, full0 + 8 * stage,
                                                                           empty0 + 8 * stage, phase ^ 1u, t, pol);
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        }
    } else {
        // ---------------- consumers.  Thread (d, j): direction term d = 2 mu + (0 fwd | 1 bwd) at
        // site slot j of the tile; its operand offsets inside a stage never change.
        const int tid = threadIdx.x;
        const int d = tid / NS, j = tid & (NS - 1);
        const int mu = d >> 1;
        const bool bwd = (d & 1) != 0;
        int loff, xoff;                                                  // element offsets in a stage
        if (mu == 0) {
            const int rt = j / L0, i = j - rt * L0;
            const int jn = rt * L0 + (bwd ? (i == 0 ? L0 - 1 : i - 1) : (i + 1 == L0 ? 0 : i + 1));
            loff = (bwd ? jn : j) * 9;
            xoff = Cfg::kXBase / SZ + jn * 3;
        } else {
            loff = ((bwd ? 3 + mu : mu) * NS + j) * 9;
            xoff = Cfg::kXBase / SZ + ((bwd ? 3 + mu : mu) * NS + j) * 3;
        }
        const bool term = d < 2 * nd;
        const T dg = (T)A.lat_diag, cf = (T)A.lat_cf, cb = (T)A.lat_cb;
        int pbuf = 0;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
            const long long row0 = (long long)t * TR;
            const int nr = (int)min((long long)TR, nrows - row0);
            const int ns = nr * L0;
            const long long row = 3 * row0 * L0 + tid;
            C ui = cmake<C>(0.0, 0.0);
            if (ROLE != ROLE_CG && tid < 3 * ns) ui = ld_ro(u + row);     // in flight while the tile lands
            mbar_wait(full0 + 8 * stage, phase);
            const C* sb = (const C*)(smem + stage * Cfg::kStageBytes);
            C* pb = part + pbuf * (9 * NS * 3);
            if (term && j < ns) {                                       // phase 1
                const C* a = sb + loff;
                const C x0 = sb[xoff], x1 = sb[xoff + 1], x2 = sb[xoff + 2];
                C v0, v1, v2;
                const C z = cmake<C>(0.0, 0.0);
                if (!bwd) {
                    v0 = cfma(a[2], x2, cfma(a[1], x1, cfma(a[0], x0, z)));
                    v1 = cfma(a[5], x2, cfma(a[4], x1, cfma(a[3], x0, z)));
                    v2 = cfma(a[8], x2, cfma(a[7], x1, cfma(a[6], x0, z)));
                } else {                                                 // U^dagger: conj of the columns
                    v0 = cfma_conj(a[6], x2, cfma_conj(a[3], x1, cfma_conj(a[0], x0, z)));
                    v1 = cfma_conj(a[7], x2, cfma_conj(a[4], x1, cfma_conj(a[1], x0, z)));
                    v2 = cfma_conj(a[8], x2, cfma_conj(a[5], x1, cfma_conj(a[2], x0, z)));
                }
                C* po = pb + (d * NS + j) * 3;
                po[0] = v0; po[1] = v1; po[2] = v2;
                if (d == 0) {                                            // keep x(s) for the diagonal term
                    const C* xs = sb + Cfg::kXBase / SZ + j * 3;
                    C* px = pb + (8 * NS + j) * 3;
                    px[0] = xs[0]; px[1] = xs[1]; px[2] = xs[2];
                }
            }
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * stage);        // this warp no longer reads the stage
            asm volatile("bar.sync 1, %0;" ::"n"(NCT) : "memory");       // partials visible
            if (tid < 3 * ns) {                                         // phase 2: scalar row 3 site0 + tid
                C f = cmake<C>(0.0, 0.0), g = f;
                for (int m = 0; m < nd; ++m) {
                    f = cadd(f, pb[(2 * m) * NS * 3 + tid]);
                    g = cadd(g, pb[(2 * m + 1) * NS * 3 + tid]);
                }
                const C xi = pb[8 * NS * 3 + tid];
                const C sum = lat_combine(dg, xi, cf, f, cb, g);
                y[row] = sum;
                lat_epilogue<C, ROLE>(acc, sum, xi, ui);
            }
            pbuf ^= 1;
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
    }
    write_partials<NACC>(st, acc);
}

// ------------------------------------------------------------------------------------------
// Warp-per-tile variant (the shipped one).  k_spmv_lat_tma above is bound by shared-memory
// bandwidth: 28 KB of its 120 KB per tile are the 3-vector partials that go from phase 1 to phase 2.
// Here ONE warp owns a tile (lane = site slot) and accumulates all 2d terms of its site in
// registers: no partials, no barrier.  A CTA is W consumer warps + the producer warp around one
// ring of STAGES stages; tile k of the CTA lives in stage k % STAGES and is consumed by warp k % W.
// ------------------------------------------------------------------------------------------
template <typename E, int W, int PW> struct LatWarpCfg {
    static constexpr int NS = 32;                                       // sites per tile = lanes
    static constexpr int kThreadsTotal = (W + PW) * 32;                  // W consumer + PW producer warps
    static constexpr int kLinkSlot = NS * 9 * (int)sizeof(E);
    static constexpr int kXSlot = NS * 3 * (int)sizeof(E);
    static constexpr int kXBase = 7 * kLinkSlot;
    static constexpr int kStageBytes = 7 * (kLinkSlot + kXSlot);
    static constexpr int smem_bytes(int stages) { return stages * kStageBytes + 2 * stages * 8; }
};

template <typename C, bool DAGGER>
__device__ __forceinline__ void lat_matvec_acc(const C* a, const C* xv, C& s0, C& s1, C& s2) {
    const C x0 = xv[0], x1 = xv[1], x2 = xv[2];
    if (!DAGGER) {
        s0 = cfma(a[2], x2, cfma(a[1], x1, cfma(a[0], x0, s0)));
        s1 = cfma(a[5], x2, cfma(a[4], x1, cfma(a[3], x0, s1)));
        s2 = cfma(a[8], x2, cfma(a[7], x1, cfma(a[6], x0, s2)));
    } else {                                                            // U^dagger: conj of the columns
        s0 = cfma_conj(a[6], x2, cfma_conj(a[3], x1, cfma_conj(a[0], x0, s0)));
        s1 = cfma_conj(a[7], x2, cfma_conj(a[4], x1, cfma_conj(a[1], x0, s1)));
        s2 = cfma_conj(a[8], x2, cfma_conj(a[5], x1, cfma_conj(a[2], x0, s2)));
    }
}

template <typename E, int W, int PW, int STAGES, int ROLE>
__global__ void __launch_bounds__(LatWarpCfg<E, W, PW>::kThreadsTotal, 1) k_spmv_lat_warp(MatDev A, SolveState* st) {
    typedef E C;
    typedef typename RealOf<E>::type T;
    typedef LatWarpCfg<E, W, PW> Cfg;
    constexpr int NACC = RoleAcc<ROLE>::value;
    constexpr int NS = Cfg::NS;
    constexpr int SZ = (int)sizeof(C);
    static_assert(STAGES % W == 0 && STAGES % PW == 0, "each stage has one producer and one consumer warp");
    if (ROLE != ROLE_GEN && st->res.done) return;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::kStageBytes);
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
        mbar_fence_init();
    }
    __syncthreads();
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    const int nd = A.lat_ndim;
    const int L0 = A.lat_ext[0];
    const int TR = A.lat_rows_per_tile;
    const long long vol = A.lat_vol;
    const long long nrows = vol / L0;
    const int ntiles = A.aux_count;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    if (warp >= W) {
        // ---------------- producer warps: one elected lane each; producer p issues the CTA's tiles p, p+PW, ...
        if (lane == 0) {
            const C* __restrict__ links = (const C*)A.val;
            const uint64_t pol = policy_evict_normal();
            const LatGeom G = lat_geom(A);
            // a stage is always filled by the same producer (stage % PW) and drained by the same
            // consumer warp (stage % W): its uses are then waited for in order by ONE thread on either
            // side, which is what the parity waits of an mbarrier need
            for (int m = 0;; ++m) {
                bool more = true;
                for (int stage = warp - W; stage < STAGES; stage += PW) {
                    const long long tl = (long long)blockIdx.x + (long long)(m * STAGES + stage) * gridDim.x;
                    if (tl >= ntiles) { more = false; break; }
                    lat_issue_tile<C, Cfg::kLinkSlot, Cfg::kXSlot, Cfg::kXBase>(G, links, x, smem + stage * Cfg::kStageBytes, full0 + 8 * stage,
                                                                               empty0 + 8 * stage, ((uint32_t)m & 1u) ^ 1u, (int)tl, pol);
                }
                if (!more) break;
            }
        }
    } else {
        // ---------------- consumer warp: lane = site slot of the tile
        const int rt = lane / L0, i0 = lane - rt * L0;
        const int jf = rt * L0 + (i0 + 1 == L0 ? 0 : i0 + 1);          // mu = 0 neighbours: same row, rotated
        const int jb = rt * L0 + (i0 == 0 ? L0 - 1 : i0 - 1);
        const T dg = (T)A.lat_diag, cf = (T)A.lat_cf, cb = (T)A.lat_cb;
        const C z = cmake<C>(0.0, 0.0);
        for (int k = warp;; k += W) {                                // k = m * (STAGES / W) * W + ... : walk own stages
            const int per = STAGES / W;                                // stages owned by this warp
            const int m = (k / W) / per, stage = warp + ((k / W) % per) * W;
            const long long tl = (long long)blockIdx.x + (long long)(m * STAGES + stage) * gridDim.x;
            if (tl >= ntiles) break;
            const uint32_t phase = (uint32_t)m & 1u;
            const long long row0 = tl * TR;
            const int nr = (int)min((long long)TR, nrows - row0);
            const int ns = nr * L0;
            const bool on = lane < ns;
            const long long row = 3 * (row0 * L0 + lane);
            C u0 = z, u1 = z, u2 = z;
            if (ROLE != ROLE_CG && on) { u0 = ld_ro(u + row); u1 = ld_ro(u + row + 1); u2 = ld_ro(u + row + 2); }
            mbar_wait(full0 + 8 * stage, phase);
            if (on) {
                const C* sb = (const C*)(smem + stage * Cfg::kStageBytes);
                const C* xs = sb + Cfg::kXBase / SZ;
                C f0 = z, f1 = z, f2 = z, g0 = z, g1 = z, g2 = z;
                lat_matvec_acc<C, false>(sb + lane * 9, xs + jf * 3, f0, f1, f2);
                lat_matvec_acc<C, true>(sb + jb * 9, xs + jb * 3, g0, g1, g2);
#pragma unroll
                for (int mu = 1; mu < 4; ++mu) {
                    if (mu >= nd) break;
                    lat_matvec_acc<C, false>(sb + (mu * NS + lane) * 9, xs + (mu * NS + lane) * 3, f0, f1, f2);
                    lat_matvec_acc<C, true>(sb + ((3 + mu) * NS + lane) * 9, xs + ((3 + mu) * NS + lane) * 3, g0, g1, g2);
                }
                const C x0 = xs[lane * 3], x1 = xs[lane * 3 + 1], x2 = xs[lane * 3 + 2];
                const C y0 = lat_combine(dg, x0, cf, f0, cb, g0);
                const C y1 = lat_combine(dg, x1, cf, f1, cb, g1);
                const C y2 = lat_combine(dg, x2, cf, f2, cb, g2);
                y[row] = y0; y[row + 1] = y1; y[row + 2] = y2;
                lat_epilogue<C, ROLE>(acc, y0, x0, u0);
                lat_epilogue<C, ROLE>(acc, y1, x1, u1);
                lat_epilogue<C, ROLE>(acc, y2, x2, u2);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * stage);            // the tile's operands are in registers
        }
    }
    write_partials<NACC>(st, acc);
}

// ------------------------------------------------------------------------------------------
// Hybrid tile kernel: two operand paths out of L2.  The all-TMA kernels above stop at ~10 TB/s of
// L2 -> shared-memory traffic (every link twice, x seven times), not at HBM.  Here only the tile's
// forward links and its own x come by bulk copy (d + 1 copies per tile instead of 14); the backward
// links U_mu(s - mu) and the neighbours' x for mu >= 1 are loaded by the consumer lanes through
// L1/L2 -- the neighbour of an x0-row is an x0-row, so a warp's loads cover contiguous ranges --
// and are issued BEFORE the warp waits for its stage.  mu = 0 neighbours: the tile's own rows rotated.
// Warp per tile, lane = site, one producer thread; a stage is owned by one consumer warp.
// ------------------------------------------------------------------------------------------
template <typename E, int W> struct LatHybCfg {
    static constexpr int NS = 32;
    static constexpr int kThreadsTotal = (W + 1) * 32;
    static constexpr int kLinkSlot = NS * 9 * (int)sizeof(E);
    static constexpr int kXSlot = NS * 3 * (int)sizeof(E);
    static constexpr int kXBase = 4 * kLinkSlot;
    static constexpr int kStageBytes = 4 * kLinkSlot + kXSlot;
    static constexpr int smem_bytes(int stages) { return stages * kStageBytes + 2 * stages * 8; }
};

template <typename E, int W, int STAGES, int ROLE>
__global__ void __launch_bounds__(LatHybCfg<E, W>::kThreadsTotal, 1) k_spmv_lat_hyb(MatDev A, SolveState* st) {
    typedef E C;
    typedef typename RealOf<E>::type T;
    typedef LatHybCfg<E, W> Cfg;
    constexpr int NACC = RoleAcc<ROLE>::value;
    constexpr int SZ = (int)sizeof(C);
    static_assert(STAGES % W == 0, "each stage has one consumer warp");
    if (ROLE != ROLE_GEN && st->res.done) return;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::kStageBytes);
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
        mbar_fence_init();
    }
    __syncthreads();
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    const C* __restrict__ links = (const C*)A.val;
    const int nd = A.lat_ndim;
    const int L0 = A.lat_ext[0];
    const int TR = A.lat_rows_per_tile;
    const long long vol = A.lat_vol;
    const int nrows = (int)(vol / L0);
    const int ntiles = A.aux_count;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    if (warp >= W) {
        if (lane == 0) {                                               // producer: d + 1 bulk copies per tile
            const uint64_t pol = policy_evict_normal();                // forward links are re-read as backward links
            for (int m = 0;; ++m) {
                bool more = true;
                for (int stage = 0; stage < STAGES; ++stage) {
                    const long long tl = (long long)blockIdx.x + (long long)(m * STAGES + stage) * gridDim.x;
                    if (tl >= ntiles) { more = false; break; }
                    const int row0 = (int)tl * TR;
                    const int nr = min(TR, nrows - row0);
                    const long long site0 = (long long)row0 * L0;
                    const uint32_t ns = (uint32_t)(nr * L0);
                    unsigned char* sb = smem + stage * Cfg::kStageBytes;
                    const uint32_t bar = full0 + 8 * stage;
                    mbar_wait(empty0 + 8 * stage, ((uint32_t)m & 1u) ^ 1u);
                    mbar_expect_tx(bar, ns * (uint32_t)SZ * (uint32_t)(9 * nd + 3));
                    for (int mu = 0; mu < nd; ++mu)
                        bulk_g2s(smem_u32(sb + mu * Cfg::kLinkSlot), links + ((long long)mu * vol + site0) * 9, ns * 9u * SZ, bar, pol);
                    bulk_g2s(smem_u32(sb + Cfg::kXBase), x + 3 * site0, ns * 3u * SZ, bar, pol);
                }
                if (!more) break;
            }
        }
    } else {
        const int rt = lane / L0, i0 = lane - rt * L0;
        const int jf = rt * L0 + (i0 + 1 == L0 ? 0 : i0 + 1);
        const int jb = rt * L0 + (i0 == 0 ? L0 - 1 : i0 - 1);
        const T dg = (T)A.lat_diag, cf = (T)A.lat_cf, cb = (T)A.lat_cb;
        const C z = cmake<C>(0.0, 0.0);
        constexpr int per = STAGES / W;
        for (int k = 0;; ++k) {
            const int m = k / per, stage = warp + (k % per) * W;
            const long long tl = (long long)blockIdx.x + (long long)(m * STAGES + stage) * gridDim.x;
            if (tl >= ntiles) break;
            const uint32_t phase = (uint32_t)m & 1u;
            const int row0 = (int)tl * TR;
            const int nr = min(TR, nrows - row0);
            const int ns = nr * L0;
            const bool on = lane < ns;
            const long long s = (long long)row0 * L0 + lane;
            const long long row = 3 * s;
            C f0 = z, f1 = z, f2 = z, g0 = z, g1 = z, g2 = z;
            C u0 = z, u1 = z, u2 = z;
            // operands that do not come through the stage: issued before the wait
            C xf[3][3], xb[3][3], ub[3][9];
            if (on) {
                if (ROLE != ROLE_CG) { u0 = ld_ro(u + row); u1 = ld_ro(u + row + 1); u2 = ld_ro(u + row + 2); }
                unsigned rem = (unsigned)(row0 + rt);
                long long str = L0;
#pragma unroll
                for (int mu = 1; mu < 4; ++mu) {
                    if (mu >= nd) break;
                    const unsigned L = (unsigned)A.lat_ext[mu];
                    const unsigned c = rem % L;
                    rem /= L;
                    const long long sf = s + (c + 1 == L ? -(long long)(L - 1) * str : str);
                    const long long sbk = s + (c == 0 ? (long long)(L - 1) * str : -str);
                    const C* pf = x + 3 * sf;
                    const C* pb = x + 3 * sbk;
                    const C* pu = links + ((long long)mu * vol + sbk) * 9;
#pragma unroll
                    for (int q = 0; q < 3; ++q) { xf[mu - 1][q] = ld_ro(pf + q); xb[mu - 1][q] = ld_ro(pb + q); }
#pragma unroll
                    for (int q = 0; q < 9; ++q) ub[mu - 1][q] = ld_ro(pu + q);
                    str *= L;
                }
            }
            mbar_wait(full0 + 8 * stage, phase);
            if (on) {
                const C* sbp = (const C*)(smem + stage * Cfg::kStageBytes);
                const C* xs = sbp + Cfg::kXBase / SZ;
                lat_matvec_acc<C, false>(sbp + lane * 9, xs + jf * 3, f0, f1, f2);
                lat_matvec_acc<C, true>(sbp + jb * 9, xs + jb * 3, g0, g1, g2);
#pragma unroll
                for (int mu = 1; mu < 4; ++mu) {
                    if (mu >= nd) break;
                    lat_matvec_acc<C, false>(sbp + (mu * Cfg::NS + lane) * 9, xf[mu - 1], f0, f1, f2);
                    lat_matvec_acc<C, true>(ub[mu - 1], xb[mu - 1], g0, g1, g2);
                }
                const C x0 = xs[lane * 3], x1 = xs[lane * 3 + 1], x2 = xs[lane * 3 + 2];
                const C y0 = lat_combine(dg, x0, cf, f0, cb, g0);
                const C y1 = lat_combine(dg, x1, cf, f1, cb, g1);
                const C y2 = lat_combine(dg, x2, cf, f2, cb, g2);
                y[row] = y0; y[row + 1] = y1; y[row + 2] = y2;
                lat_epilogue<C, ROLE>(acc, y0, x0, u0);
                lat_epilogue<C, ROLE>(acc, y1, x1, u1);
                lat_epilogue<C, ROLE>(acc, y2, x2, u2);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * stage);
        }
    }
    write_partials<NACC>(st, acc);
}

// ------------------------------------------------------------------------------------------
// Blocked tile kernel (round 2).  The all-TMA kernels above move 84 elements per site from L2 into shared memory
// (7 link rows and 7 x rows per x0-row) and stop at the L2 -> SM rate, not at HBM.  Here a tile is a block of
// R1 x R2 x0-rows in the (x1, x2) plane at fixed x3: inside the block the backward link U_mu(s - mu) of a row is
// the forward link of the neighbouring row and the neighbours' x are the neighbouring rows' own x, both already
// staged, so only the block's surface comes in addition:
//   link rows per tile: 4 R1 R2 (forward) + R2 (mu = 1, row x1 - 1) + R1 (mu = 2, row x2 - 1) + R1 R2 (mu = 3)
//   x rows per tile:    R1 R2 (own) + 2 R2 (x1 -+ 1) + 2 R1 (x2 -+ 1) + 2 R1 R2 (x3 -+ 1)
// 2 x 2: 69 elements per site instead of 84, and 25 bulk copies per 128 sites instead of 56 (R1 consecutive
// x1-rows are one contiguous range).  One consumer warp per row of the block (lane = x0, so L0 = 32), every
// operand out of shared memory, the same order of multiply-adds as k_spmv_lat_warp (bit-identical y); a stage is
// filled by one producer warp (one per stage) and drained by all R1 R2 consumer warps.
// Needs 4 dimensions, L0 = 32, R1 | L1, R2 | L2 (lat_blk_supported, spmv_role.cu).
// ------------------------------------------------------------------------------------------
template <typename E, int R1, int R2, int STAGES> struct LatBlkCfg {
    static constexpr int L0 = 32;
    static constexpr int NR = R1 * R2;                                   // rows per tile = consumer warps
    static constexpr int kThreadsTotal = (NR + STAGES) * 32;             // + one producer warp per stage
    static constexpr int kLinkRow = L0 * 9 * (int)sizeof(E), kXRow = L0 * 3 * (int)sizeof(E);
    // link rows: F[mu][j][i] (4 NR), B1[j], B2[i], B3[j][i];   x rows: X[j][i], XF1[j], XB1[j], XF2[i], XB2[i], XF3, XB3
    static constexpr int oB1 = 4 * NR, oB2 = oB1 + R2, oB3 = oB2 + R1, kLinkRows = oB3 + NR;
    static constexpr int oXF1 = NR, oXB1 = oXF1 + R2, oXF2 = oXB1 + R2, oXB2 = oXF2 + R1, oXF3 = oXB2 + R1, oXB3 = oXF3 + NR,
                         kXRows = oXB3 + NR;
    static constexpr int kXBase = kLinkRows * kLinkRow;
    static constexpr int kStageBytes = kXBase + kXRows * kXRow;
    static constexpr int smem_bytes() { return STAGES * kStageBytes + 2 * STAGES * 8; }
};

template <typename E, int R1, int R2, int STAGES, int ROLE>
__global__ void __launch_bounds__((LatBlkCfg<E, R1, R2, STAGES>::kThreadsTotal), 1) k_spmv_lat_blk(MatDev A, SolveState* st) {
    typedef E C;
    typedef typename RealOf<E>::type T;
    typedef LatBlkCfg<E, R1, R2, STAGES> Cfg;
    constexpr int NACC = RoleAcc<ROLE>::value;
    constexpr int NR = Cfg::NR, L0 = Cfg::L0;
    constexpr int SZ = (int)sizeof(C);
    if (ROLE != ROLE_GEN && st->res.done) return;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::kStageBytes);
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, NR); }
        mbar_fence_init();
    }
    __syncthreads();
    const C* x; C* y; const C* u;
    role_vectors<C, ROLE>(st, x, y, u);
    const int L1 = A.lat_ext[1], L2 = A.lat_ext[2], L3 = A.lat_ext[3];
    const int nA = L1 / R1, nB = L2 / R2;
    const int ntiles = nA * nB * L3;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    if (warp >= NR) {
        // ---------------- producer warp p fills stage p: tiles blockIdx.x + (m STAGES + p) gridDim.x
        if (lane == 0) {
            const int stage = warp - NR;
            const C* __restrict__ links = (const C*)A.val;
            const uint64_t pol = policy_evict_normal();
            const long long vol = A.lat_vol;
            unsigned char* sb = smem + stage * Cfg::kStageBytes;
            const uint32_t bar = full0 + 8 * stage, ebar = empty0 + 8 * stage;
            const uint32_t lrows = (uint32_t)(R1 * Cfg::kLinkRow), xrows = (uint32_t)(R1 * Cfg::kXRow);
            for (int m = 0;; ++m) {
                const long long tl = (long long)blockIdx.x + (long long)(m * STAGES + stage) * gridDim.x;
                if (tl >= ntiles) break;
                const int a = (int)(tl % nA), b = (int)((tl / nA) % nB), x3 = (int)(tl / ((long long)nA * nB));
                const int x1 = a * R1, x2 = b * R2;
                const int x1m = x1 == 0 ? L1 - 1 : x1 - 1, x1p = x1 + R1 == L1 ? 0 : x1 + R1;
                const int x2m = x2 == 0 ? L2 - 1 : x2 - 1, x2p = x2 + R2 == L2 ? 0 : x2 + R2;
                const int x3m = x3 == 0 ? L3 - 1 : x3 - 1, x3p = x3 + 1 == L3 ? 0 : x3 + 1;
                // first site of x0-row (c1, c2, c3); link / x row `slot` of the stage
#define MSOLVE_SITE0(c1, c2, c3) ((long long)L0 * ((c1) + (long long)L1 * ((c2) + (long long)L2 * (c3))))
#define MSOLVE_LROW(slot) smem_u32(sb + (slot) * Cfg::kLinkRow)
#define MSOLVE_XROW(slot) smem_u32(sb + Cfg::kXBase + (slot) * Cfg::kXRow)
                mbar_wait(ebar, ((uint32_t)m & 1u) ^ 1u);
                mbar_expect_tx(bar, (uint32_t)Cfg::kStageBytes);
#pragma unroll
                for (int j = 0; j < R2; ++j) {
                    const long long s0 = MSOLVE_SITE0(x1, x2 + j, x3);
#pragma unroll
                    for (int mu = 0; mu < 4; ++mu)
                        bulk_g2s(MSOLVE_LROW(mu * NR + j * R1), links + ((long long)mu * vol + s0) * 9, lrows, bar, pol);
                    bulk_g2s(MSOLVE_XROW(j * R1), x + 3 * s0, xrows, bar, pol);
                    const long long s1m = MSOLVE_SITE0(x1m, x2 + j, x3), s1p = MSOLVE_SITE0(x1p, x2 + j, x3);
                    bulk_g2s(MSOLVE_LROW(Cfg::oB1 + j), links + (1ll * vol + s1m) * 9, (uint32_t)Cfg::kLinkRow, bar, pol);
                    bulk_g2s(MSOLVE_XROW(Cfg::oXF1 + j), x + 3 * s1p, (uint32_t)Cfg::kXRow, bar, pol);
                    bulk_g2s(MSOLVE_XROW(Cfg::oXB1 + j), x + 3 * s1m, (uint32_t)Cfg::kXRow, bar, pol);
                    const long long s3m = MSOLVE_SITE0(x1, x2 + j, x3m), s3p = MSOLVE_SITE0(x1, x2 + j, x3p);
                    bulk_g2s(MSOLVE_LROW(Cfg::oB3 + j * R1), links + (3ll * vol + s3m) * 9, lrows, bar, pol);
                    bulk_g2s(MSOLVE_XROW(Cfg::oXF3 + j * R1), x + 3 * s3p, xrows, bar, pol);
                    bulk_g2s(MSOLVE_XROW(Cfg::oXB3 + j * R1), x + 3 * s3m, xrows, bar, pol);
                }
                const long long s2m = MSOLVE_SITE0(x1, x2m, x3), s2p = MSOLVE_SITE0(x1, x2p, x3);
                bulk_g2s(MSOLVE_LROW(Cfg::oB2), links + (2ll * vol + s2m) * 9, lrows, bar, pol);
                bulk_g2s(MSOLVE_XROW(Cfg::oXF2), x + 3 * s2p, xrows, bar, pol);
                bulk_g2s(MSOLVE_XROW(Cfg::oXB2), x + 3 * s2m, xrows, bar, pol);
#undef MSOLVE_SITE0
#undef MSOLVE_LROW
#undef MSOLVE_XROW
            }
        }
    } else {
        // ---------------- consumer warp = row (i, j) of the block, lane = x0
        const int i = warp % R1, j = warp / R1, r = warp;
        const int jf = lane + 1 == L0 ? 0 : lane + 1, jb = lane == 0 ? L0 - 1 : lane - 1;
        const T dg = (T)A.lat_diag, cf = (T)A.lat_cf, cb = (T)A.lat_cb;
        const C z = cmake<C>(0.0, 0.0);
        // operand rows of this warp inside a stage (in units of C): a neighbour inside the block, else the surface row
        constexpr int LR = L0 * 9, XR = L0 * 3, XB = Cfg::kXBase / SZ;
        const int l1b = (i > 0 ? (1 * NR + r - 1) : (Cfg::oB1 + j)) * LR;
        const int l2b = (j > 0 ? (2 * NR + r - R1) : (Cfg::oB2 + i)) * LR;
        const int x1f = XB + (i + 1 < R1 ? r + 1 : Cfg::oXF1 + j) * XR, x1b = XB + (i > 0 ? r - 1 : Cfg::oXB1 + j) * XR;
        const int x2f = XB + (j + 1 < R2 ? r + R1 : Cfg::oXF2 + i) * XR, x2b = XB + (j > 0 ? r - R1 : Cfg::oXB2 + i) * XR;
        for (int k = 0;; ++k) {
            const int stage = k % STAGES, m = k / STAGES;
            const long long tl = (long long)blockIdx.x + (long long)k * gridDim.x;
            if (tl >= ntiles) break;
            const int a = (int)(tl % nA), b = (int)((tl / nA) % nB), x3 = (int)(tl / ((long long)nA * nB));
            const long long row = 3 * ((long long)L0 * ((a * R1 + i) + (long long)L1 * ((b * R2 + j) + (long long)L2 * x3)) + lane);
            C u0 = z, u1 = z, u2 = z;
            if (ROLE != ROLE_CG) { u0 = ld_ro(u + row); u1 = ld_ro(u + row + 1); u2 = ld_ro(u + row + 2); }
            mbar_wait(full0 + 8 * stage, (uint32_t)m & 1u);
            const C* sb = (const C*)(smem + stage * Cfg::kStageBytes);
            C f0 = z, f1 = z, f2 = z, g0 = z, g1 = z, g2 = z;
            lat_matvec_acc<C, false>(sb + r * LR + lane * 9, sb + XB + r * XR + jf * 3, f0, f1, f2);
            lat_matvec_acc<C, true>(sb + r * LR + jb * 9, sb + XB + r * XR + jb * 3, g0, g1, g2);
            lat_matvec_acc<C, false>(sb + (1 * NR + r) * LR + lane * 9, sb + x1f + lane * 3, f0, f1, f2);
            lat_matvec_acc<C, true>(sb + l1b + lane * 9, sb + x1b + lane * 3, g0, g1, g2);
            lat_matvec_acc<C, false>(sb + (2 * NR + r) * LR + lane * 9, sb + x2f + lane * 3, f0, f1, f2);
            lat_matvec_acc<C, true>(sb + l2b + lane * 9, sb + x2b + lane * 3, g0, g1, g2);
            lat_matvec_acc<C, false>(sb + (3 * NR + r) * LR + lane * 9, sb + XB + (Cfg::oXF3 + r) * XR + lane * 3, f0, f1, f2);
            lat_matvec_acc<C, true>(sb + (Cfg::oB3 + r) * LR + lane * 9, sb + XB + (Cfg::oXB3 + r) * XR + lane * 3, g0, g1, g2);
            const C* xo = sb + XB + r * XR + lane * 3;
            const C x0 = xo[0], x1 = xo[1], x2 = xo[2];
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * stage);            // the tile's operands are in registers
            const C y0 = lat_combine(dg, x0, cf, f0, cb, g0);
            const C y1 = lat_combine(dg, x1, cf, f1, cb, g1);
            const C y2 = lat_combine(dg, x2, cf, f2, cb, g2);
            y[row] = y0; y[row + 1] = y1; y[row + 2] = y2;
            lat_epilogue<C, ROLE>(acc, y0, x0, u0);
            lat_epilogue<C, ROLE>(acc, y1, x1, u1);
            lat_epilogue<C, ROLE>(acc, y2, x2, u2);
        }
    }
    write_partials<NACC>(st, acc);
}

}  // namespace msolve
