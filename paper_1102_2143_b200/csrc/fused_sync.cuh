// fused_sync.cuh -- what the cooperative whole-solve kernels (fused_small.cu, resident.cu) share: the combined
// grid barrier + sum, the header staged in shared memory, the result written back by CTA 0.
#pragma once

#include "common.cuh"

namespace msolve {

// per-CTA private state at the start of the dynamic shared memory of a whole-solve kernel: recurrences, result block,
// header, per-system norms; what follows it is 16-byte aligned
constexpr int kFusedOffRes = (int)sizeof(Recur);
constexpr int kFusedOffHdr = kFusedOffRes + (int)sizeof(SolveResult);
constexpr int kFusedOffNorm = kFusedOffHdr + (int)sizeof(SolveHeader);
constexpr int kFusedFixedBytes = (kFusedOffNorm + (int)sizeof(double) * kMaxShifts + 15) / 16 * 16;

// ---- grid-wide barrier and sum in ONE round trip to L2.  Every CTA publishes its share of the sum as 64-bit words
// that each carry half a double and the generation of the barrier (8-byte stores are single-copy atomic, so a word
// is either old or complete); every CTA polls the words of all CTAs (spread over its threads) until they carry the
// current generation -- the same load that detects the arrival delivers the value -- and adds the shares in CTA
// order: the same fixed-order tree in every CTA, so every CTA holds the same bits.  There is no atomic and no single
// counter all CTAs serialise on (148 CTAs on one L2 atomic cost ~2 us per barrier).  Release / acquire: a fence
// before the words are stored, a fence after the last one has been seen.  Slots are double-buffered by the parity of
// the generation: a CTA can only overwrite its slot of generation g at generation g + 2, which it reaches only after
// every CTA has passed g + 1, i.e. has finished reading generation g.
__device__ __forceinline__ void st_relaxed_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// NACC = 0: barrier only.  acc: this thread's share (in); out: the grid-wide sums (the same in every thread).
template <int NACC>
__device__ __forceinline__ void fused_allreduce(SolveState* st, unsigned long long& gen, double* acc, double* out, double* red) {
    ++gen;
    const unsigned g32 = (unsigned)gen;
    FusedSlot* slots = st->fslot[gen & 1ull];
    __shared__ double bc[kAccMax];
    __shared__ unsigned s_lo[kFusedMaxCtas * 2 * kAccMax];
    const int ncta = (int)gridDim.x;
    __syncthreads();                         // everything this CTA wrote so far is ordered before the fence below
    if constexpr (NACC > 0) {
        double a[NACC];
#pragma unroll
        for (int i = 0; i < NACC; ++i) a[i] = acc[i];
        block_sum<NACC>(a, red);
        if (threadIdx.x == 0) {
            __threadfence();
#pragma unroll
            for (int i = 0; i < NACC; ++i) {
                const unsigned long long bits = (unsigned long long)__double_as_longlong(a[i]);
                st_relaxed_u64(&slots[blockIdx.x].w[2 * i], ((unsigned long long)g32 << 32) | (bits & 0xffffffffull));
                st_relaxed_u64(&slots[blockIdx.x].w[2 * i + 1], ((unsigned long long)g32 << 32) | (bits >> 32));
            }
        }
        for (int j = threadIdx.x; j < ncta * 2 * NACC; j += blockDim.x) {
            const int c = j / (2 * NACC), k = j - c * 2 * NACC;
            unsigned long long v;
            do { v = ld_relaxed_u64(&slots[c].w[k]); } while ((unsigned)(v >> 32) != g32);
            s_lo[j] = (unsigned)v;
        }
    } else {
        if (threadIdx.x == 0) { __threadfence(); st_relaxed_u64(&slots[blockIdx.x].tag, gen); }
        for (int c = threadIdx.x; c < ncta; c += blockDim.x)
            while (ld_relaxed_u64(&slots[c].tag) != gen) {}
    }
    __threadfence();
    __syncthreads();                         // every CTA has arrived; their writes are visible to this CTA
    if constexpr (NACC > 0) {
        double a[NACC];
#pragma unroll
        for (int i = 0; i < NACC; ++i) a[i] = 0.0;
        for (int c = threadIdx.x; c < ncta; c += blockDim.x) {
#pragma unroll
            for (int i = 0; i < NACC; ++i)
                a[i] += __longlong_as_double((long long)(((unsigned long long)s_lo[(c * NACC + i) * 2 + 1] << 32) | s_lo[(c * NACC + i) * 2]));
        }
        block_sum<NACC>(a, red);
        if (threadIdx.x == 0) {
#pragma unroll
            for (int i = 0; i < NACC; ++i) bc[i] = a[i];
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < NACC; ++i) out[i] = bc[i];
    }
}

// The header (pointers, sizes, shifts) and the per-system norms of eq. (6) are read in every phase; every barrier
// invalidates L1, so they live in shared memory for the whole solve.
// The header arrives as a KERNEL ARGUMENT (no host-to-device copy before the launch).
__device__ __forceinline__ void fused_stage_header(const SolveHeader& hp, const SolveState* st, unsigned char* dst, double* rhs_norm) {
    const int* src = (const int*)&hp;
    int* d = (int*)dst;
    for (int i = threadIdx.x; i < (int)(sizeof(SolveHeader) / sizeof(int)); i += blockDim.x) d[i] = src[i];
    for (int k = threadIdx.x; k < kMaxShifts; k += blockDim.x) rhs_norm[k] = st->rhs_norm[k];
    __syncthreads();
}

__device__ __forceinline__ void fused_publish(SolveState* st, const SolveResult& res, unsigned long long gen) {
    if (blockIdx.x != 0) return;
    __syncthreads();
    if (threadIdx.x == 0) st->fused_gen = gen;
    const int* src = (const int*)&res;
    int* dst = (int*)&st->res;
    for (int i = threadIdx.x; i < (int)(sizeof(SolveResult) / sizeof(int)); i += blockDim.x) dst[i] = src[i];
}

// msolve_set_phase_clock: thread 0 of CTA 0 adds the time since the previous mark to slot i (off: one uniform branch)
struct PhaseClock {
    unsigned long long* ns;
    unsigned long long t0;
    __device__ __forceinline__ static unsigned long long now() {
        unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t;
    }
    __device__ __forceinline__ explicit PhaseClock(unsigned long long* p) : ns(blockIdx.x == 0 && threadIdx.x == 0 ? p : nullptr), t0(0) {
        if (ns) t0 = now();
    }
    __device__ __forceinline__ void mark(int i) {
        if (ns) { const unsigned long long t = now(); ns[i] += t - t0; t0 = t; }
    }
};

}  // namespace msolve
