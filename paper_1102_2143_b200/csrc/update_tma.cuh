// update_tma.cuh -- the fused multishift update of CG-M (Alg. 1 l.21, 24, 28,
// 29) with every byte moved by the TMA engine.
//
// Same arithmetic and operand order as k_cgm_update (kernels.cuh): per element
//   p_k <- zeta_k r + alpha_k p_k (lagged l.29) ; x_k <- x_k - beta_k p_k (l.28) for every active
//   shift, then r <- r + beta Ap (l.21) and |r|^2 (l.24).
// What differs is the data movement.  The register version keeps 8 loads of 16 bytes in flight per
// thread (65 KB per SM); here one CTA per SM owns a ring of STAGES shared-memory stages and a
// producer thread streams "items" into it with 1-D bulk async copies:
//   item 0 of a tile   = (r, Ap) of TILE packs,
//   item 1+a of a tile = (x_k, p_k) of the a-th active shift.
// Consumer warp w owns packs [w*TILE/8, (w+1)*TILE/8) of every item: it reads them from shared
// memory, writes the results back IN PLACE and stores its slice with bulk async copies
// (shared -> global, bulk_group completion), so up to STAGES * 32 KB per SM are in flight whatever
// the register budget is.  A stage goes back to the producer once the stores of the item LAG items
// earlier have finished READING shared memory (cp.async.bulk.wait_group.read).
// Measured on B200 (config 4, 16 shifts): 1.1235 ms per launch against 1.1237 ms for the register
// kernel -- two unrelated ways of moving the bytes end at the same 6.0 TB/s, which is therefore the
// HBM3e ceiling for this 51 % read / 49 % write mix, not a property of either kernel.  The register
// kernel stays the default; this one is selected with MSOLVE_CFG_UPDATE_KERNEL = 1.
#pragma once

#include "kernels.cuh"
#include "spmv.cuh"

namespace msolve {

// shared -> global bulk copy of this thread's bulk async-group
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src, uint32_t bytes, uint64_t policy) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                 ::"l"(dst), "r"(src), "r"(bytes), "l"(policy) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <typename E> struct UpdTmaCfg {
    static constexpr int VEC = 16 / (int)sizeof(E);        // elements per 16-byte pack
    static constexpr int kWarps = 8;                       // consumer warps
    static constexpr int kConsumers = kWarps * 32;
    static constexpr int kThreadsTotal = kConsumers + 32;
    static constexpr int kTile = 1024;                     // packs per tile (16 KB per vector)
    static constexpr int kPpl = kTile / kConsumers;        // packs per lane
    static constexpr int kVecBytes = kTile * 16;
    static constexpr int kStageBytes = 2 * kVecBytes;      // (r, Ap) or (x_k, p_k)
    static constexpr int smem_bytes(int stages) { return stages * kStageBytes + 2 * stages * 8; }
};

template <typename E, int STAGES, int LAG>
__global__ void __launch_bounds__(UpdTmaCfg<E>::kThreadsTotal, 1) k_cgm_update_tma(SolveState* st) {
    if (st->res.done) return;
    typedef E C;
    typedef typename RealOf<E>::type T;
    typedef UpdTmaCfg<E> Cfg;
    constexpr int VEC = Cfg::VEC;
    typedef Pack<E, VEC> P;
    static_assert(LAG >= 1 && LAG < STAGES - 1, "need at least one stage free for loads");
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::kStageBytes);
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
    __shared__ T s_zeta[kMaxShifts], s_alpha[kMaxShifts], s_beta[kMaxShifts];
    __shared__ int s_k[kMaxShifts];
    const int na = st->res.nactive;
    const bool first = st->res.n_iter == 0;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        s_k[a] = st->rc.active[a];
        s_zeta[a] = (T)st->rc.coef[3 * a + 0];
        s_alpha[a] = (T)st->rc.coef[3 * a + 1];
        s_beta[a] = (T)st->rc.coef[3 * a + 2];
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, Cfg::kWarps); }
        mbar_fence_init();
    }
    __syncthreads();
    const long long n = st->h.n, nvec = n / VEC, pks = st->h.pk_stride;
    const int ntiles = (int)((nvec + Cfg::kTile - 1) / Cfg::kTile);
    unsigned char* r = (unsigned char*)st->h.r;
    const unsigned char* q = (const unsigned char*)st->h.q;
    unsigned char* x = (unsigned char*)st->h.x;
    unsigned char* pk = (unsigned char*)st->h.pk;
    const long long xstride = st->h.x_stride * (long long)sizeof(E), pstride = pks * (long long)sizeof(E);
    double acc[1] = {0.0};
    int stage = 0;
    uint32_t phase = 0;
    if (threadIdx.x >= Cfg::kConsumers) {
        // ---------------- producer: one elected lane of the last warp
        if (threadIdx.x == Cfg::kConsumers) {
            const uint64_t pol = policy_evict_first(), polr = policy_evict_normal();
            for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
                const long long p0 = (long long)t * Cfg::kTile;
                const uint32_t bytes = (uint32_t)min((long long)Cfg::kTile, nvec - p0) * 16u;
                const long long off = p0 * 16;
                for (int item = 0; item <= na; ++item) {
                    mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                    const uint32_t sb = smem_u32(smem + stage * Cfg::kStageBytes);
                    const uint32_t bar = full0 + 8 * stage;
                    if (item == 0) {
                        mbar_expect_tx(bar, 2 * bytes);
                        bulk_g2s(sb, r + off, bytes, bar, polr);
                        bulk_g2s(sb + Cfg::kVecBytes, q + off, bytes, bar, pol);
                    } else if (!first) {
                        const int k = s_k[item - 1];
                        mbar_expect_tx(bar, 2 * bytes);
                        bulk_g2s(sb, x + k * xstride + off, bytes, bar, pol);
                        bulk_g2s(sb + Cfg::kVecBytes, pk + k * pstride + off, bytes, bar, pol);
                    } else {
                        mbar_arrive(bar);                         // x_k = 0, p_k = b: nothing to load
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else {
        // ---------------- consumers: warp w owns packs [w*SL, (w+1)*SL) of every item
        constexpr int SL = Cfg::kTile / Cfg::kWarps;              // packs per warp slice
        constexpr int PPL = SL / 32;                              // packs per lane
        const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
        const T beta = (T)st->rc.beta.re;
        const uint64_t pol = policy_evict_first(), polr = policy_evict_normal();
        int rel_stage = 0;                                        // next stage to hand back (LAG items behind)
        long long items = 0;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
            const long long p0 = (long long)t * Cfg::kTile;
            const int cnt = (int)min((long long)Cfg::kTile, nvec - p0);        // packs in this tile
            const int sl_cnt = max(0, min(SL, cnt - warp * SL));                // packs in this warp's slice
            const long long sl_off = (p0 + warp * SL) * 16;                      // byte offset of the slice in a vector
            P rv[PPL];
            for (int item = 0; item <= na; ++item) {
                mbar_wait(full0 + 8 * stage, phase);
                unsigned char* sb = smem + stage * Cfg::kStageBytes;
                P* va = (P*)sb + warp * SL;                       // r   | x_k
                P* vb = (P*)(sb + Cfg::kVecBytes) + warp * SL;    // Ap  | p_k
                if (item == 0) {
#pragma unroll
                    for (int j = 0; j < PPL; ++j) {
                        const int i = lane + 32 * j;
                        if (i < sl_cnt) {
                            rv[j] = va[i];                        // r_n stays in registers for the shifts
                            const P qv = vb[i];
                            P rn;
#pragma unroll
                            for (int e = 0; e < VEC; ++e) {
                                rn.v[e] = caxpy_r(rv[j].v[e], beta, qv.v[e]);        // l.21
                                acc[0] += cnorm2(rn.v[e]);                           // l.24
                            }
                            va[i] = rn;
                        }
                    }
                    fence_async_smem();
                    __syncwarp();
                    if (lane == 0 && sl_cnt > 0) bulk_s2g(r + sl_off, smem_u32(va), (uint32_t)sl_cnt * 16u, polr);
                } else {
                    const int k = s_k[item - 1];
                    const T zk = s_zeta[item - 1], ak = s_alpha[item - 1], bk = s_beta[item - 1];
#pragma unroll
                    for (int j = 0; j < PPL; ++j) {
                        const int i = lane + 32 * j;
                        if (i < sl_cnt) {
                            P xv, pv;
                            if (!first) { xv = va[i]; pv = vb[i]; }
                            P xo, po;
#pragma unroll
                            for (int e = 0; e < VEC; ++e) {
                                C pe, xe;
                                if (first) { pe = rv[j].v[e]; xe = cmake<C>(0.0, 0.0); }   // p_k = b, x_k = 0
                                else {
                                    pe = clin_r(zk, rv[j].v[e], ak, pv.v[e]);              // l.29 (lagged)
                                    xe = xv.v[e];
                                }
                                xo.v[e] = caxpy_r(xe, -bk, pe);                            // l.28
                                po.v[e] = pe;
                            }
                            va[i] = xo;
                            vb[i] = po;
                        }
                    }
                    fence_async_smem();
                    __syncwarp();
                    if (lane == 0 && sl_cnt > 0) {
                        bulk_s2g(x + k * xstride + sl_off, smem_u32(va), (uint32_t)sl_cnt * 16u, pol);
                        bulk_s2g(pk + k * pstride + sl_off, smem_u32(vb), (uint32_t)sl_cnt * 16u, pol);
                    }
                }
                if (lane == 0) {
                    bulk_commit();
                    if (++items > LAG) {                          // the stores of item (items-1-LAG) have read smem
                        bulk_wait_read<LAG>();
                        mbar_arrive(empty0 + 8 * rel_stage);
                        if (++rel_stage == STAGES) rel_stage = 0;
                    }
                }
                if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            }
        }
        if (lane == 0) bulk_wait_all();                           // all stores of this warp are complete
    }
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) {
        st->partial[blockIdx.x] = acc[0];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

}  // namespace msolve
