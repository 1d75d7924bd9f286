// kernels.cuh -- vector-update and scalar-recurrence kernels of the multishift iterations.
//
// CG-M (Alg. 1):
//   k_cgm_pupdate   A1  p <- r + alpha p                                  (l.27)
//   k_cgm_scal1     A4  beta, zeta_new_k, beta_k from <p,Ap>              (l.20, 22, 23)
//   k_cgm_update    A5  fused multishift update, lagged form: per element read r, Ap once;
//                       per active shift p_k <- zeta_k r + alpha_k p_k (l.29 of the PREVIOUS
//                       iteration), x_k <- x_k - beta_k p_k (l.28); r <- r + beta Ap (l.21);
//                       |r|^2 partials (l.24)
//   k_cgm_scal2     A6  alpha, alpha_k, zeta shuffle, stop/mask test      (l.25, 26, 30, 31, 15)
// BiCGStab-M:
//   k_bi_scal1, k_bi_supdate (s = r + beta q), k_bi_scal2, k_bi_update, k_bi_scal3.
//
// The per-shift zeta/alpha/beta recurrences stay on the device; converged
// shifts are removed from the `active` list, so the update kernels never touch their vectors.
//
// Every step is a __device__ function over (header, result, recurrences): the k_* kernels below run one step each
// on the device-resident SolveState (the iteration as a graph of kernels); fused_small.cuh strings the same
// functions together inside one cooperative kernel for systems that live in L2.  `cta` / `ncta` are the CTA's
// index and the number of CTAs the elements are spread over.
#pragma once

#include "common.cuh"

namespace msolve {

// ----------------------------------------------------------------------------- vector packs
// Pack<E,VEC>: VEC elements of type E moved by ONE load/store instruction (16 bytes whenever the
// vector length allows it: 1 complex128, 2 complex64 / float64, 4 float32).
template <typename E, int VEC> struct __align__(sizeof(E) * VEC) Pack { E v[VEC]; };

// Loads / stores go through the CUDA vector type of the same size (no unions: type punning through
// memory made ptxas reuse registers between the per-shift loads and serialise them).
#define MSOLVE_PACK_IO(E, VEC, V, UNPACK, PACK)                                                     \
    template <bool STREAM> __device__ __forceinline__ Pack<E, VEC> ld_pack(const Pack<E, VEC>* p) { \
        const V t = STREAM ? __ldcs((const V*)p) : *(const V*)p;                                    \
        Pack<E, VEC> r; UNPACK; return r;                                                           \
    }                                                                                               \
    template <bool STREAM> __device__ __forceinline__ void st_pack(Pack<E, VEC>* p, const Pack<E, VEC>& r) { \
        const V t = PACK;                                                                           \
        if (STREAM) __stcs((V*)p, t); else *(V*)p = t;                                              \
    }
MSOLVE_PACK_IO(double2, 1, double2, r.v[0] = t, r.v[0])
MSOLVE_PACK_IO(float2, 1, float2, r.v[0] = t, r.v[0])
MSOLVE_PACK_IO(float2, 2, float4, (r.v[0] = make_float2(t.x, t.y), r.v[1] = make_float2(t.z, t.w)),
               make_float4(r.v[0].x, r.v[0].y, r.v[1].x, r.v[1].y))
MSOLVE_PACK_IO(double, 1, double, r.v[0] = t, r.v[0])
MSOLVE_PACK_IO(double, 2, double2, (r.v[0] = t.x, r.v[1] = t.y), make_double2(r.v[0], r.v[1]))
MSOLVE_PACK_IO(float, 1, float, r.v[0] = t, r.v[0])
MSOLVE_PACK_IO(float, 4, float4, (r.v[0] = t.x, r.v[1] = t.y, r.v[2] = t.z, r.v[3] = t.w),
               make_float4(r.v[0], r.v[1], r.v[2], r.v[3]))
#undef MSOLVE_PACK_IO

// ----------------------------------------------------------------------------- init
// r <- b, p <- b (Alg. 1 l.9-10); partial |b|^2 (l.13).  p_k <- b and x_k <- 0 (l.11-12) are not
// materialised: the first update treats them as such without reading them.
template <typename E, int VEC>
__device__ __forceinline__ double init_vectors_fn(const SolveHeader& h, int cta, int ncta) {
    typedef Pack<E, VEC> P;
    const long long nvec = h.n / VEC;
    const P* b = (const P*)h.b;
    P* r = (P*)h.r;
    P* p = (P*)h.p;
    double acc = 0.0;
    const long long stride = (long long)ncta * blockDim.x;
    for (long long i = (long long)cta * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const P bv = ld_pack<false>(b + i);
        st_pack<false>(r + i, bv);
        st_pack<false>(p + i, bv);
#pragma unroll
        for (int e = 0; e < VEC; ++e) acc += cnorm2(bv.v[e]);
    }
    return acc;
}

template <typename E, int VEC>
__global__ void __launch_bounds__(kThreads) k_init_vectors(SolveState* st) {
    double acc[1] = {init_vectors_fn<E, VEC>(st->h, blockIdx.x, gridDim.x)};
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) {
        st->partial[blockIdx.x] = acc[0];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

// Scalars of l.2-8, 13-14 and the BiCGStab-M analogue from bb = <b,b>; b = 0 ends the solve at once.
__device__ __forceinline__ void init_state_fn(const SolveHeader& h, SolveResult& res, Recur& rc, double bb) {
    const int S = h.S;
    for (int k = threadIdx.x; k < S; k += blockDim.x) {
        rc.zeta_prev[k] = {1.0, 0.0}; rc.zeta[k] = {1.0, 0.0}; rc.zeta_new[k] = {1.0, 0.0};
        rc.rho[k] = {1.0, 0.0}; rc.rho_new[k] = {1.0, 0.0};
        rc.beta_k[k] = {0.0, 0.0}; rc.alpha_k[k] = {0.0, 0.0}; rc.chi_k[k] = {0.0, 0.0};
        rc.active[k] = k;
        res.conv_iter[k] = (bb == 0.0) ? 0 : -1;
        res.relres[k] = (bb == 0.0) ? 0.0 : 1.0;
    }
    if (threadIdx.x == 0) {
        rc.alpha = {0.0, 0.0}; rc.beta = {0.0, 0.0}; rc.beta_prev = {1.0, 0.0};
        rc.delta = {bb, 0.0};            // <r0,r> = <b,b>
        rc.chi = {0.0, 0.0}; rc.alpha_new = {0.0, 0.0}; rc.delta_new = {0.0, 0.0};
        rc.R0 = bb; rc.R1 = bb; rc.bnorm = sqrt(bb);
        res.n_iter = 0;
        res.status = MSOLVE_OK;
        res.nactive = S;
        res.zero_rhs = (bb == 0.0);
        res.done = (bb == 0.0) || !isfinite(bb) || h.max_iter <= 0;
        if (!isfinite(bb)) res.status = MSOLVE_BREAKDOWN;
        else if (bb != 0.0 && h.max_iter <= 0) res.status = MSOLVE_MAXITER;
    }
    __syncthreads();
}


constexpr int kPupdUnroll = 4;   // 2 * 4 independent 16-byte loads in flight per thread
// ----------------------------------------------------------------------------- CG-M
// A1: p <- r + alpha p  (l.27; at n = 0 p = b already)
template <typename E, int VEC>
__device__ __forceinline__ void cgm_pupdate_fn(const SolveHeader& h, const Recur& rc, int cta, int ncta) {
    typedef typename RealOf<E>::type T;
    typedef Pack<E, VEC> P;
    const long long nvec = h.n / VEC;
    const P* r = (const P*)h.r;
    P* p = (P*)h.p;
    const T alpha = (T)rc.alpha.re;
    const long long stride = (long long)ncta * blockDim.x;
    constexpr int U = kPupdUnroll;
    long long i = (long long)cta * blockDim.x + threadIdx.x;
    for (; i + (U - 1) * stride < nvec; i += U * stride) {
        P rv[U], pv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { rv[u] = ld_pack<false>(r + i + u * stride); pv[u] = ld_pack<false>(p + i + u * stride); }
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int e = 0; e < VEC; ++e) pv[u].v[e] = caxpy_r(rv[u].v[e], alpha, pv[u].v[e]);
            st_pack<false>(p + i + u * stride, pv[u]);
        }
    }
    for (; i < nvec; i += stride) {
        const P rv = ld_pack<false>(r + i);
        P pv = ld_pack<false>(p + i);
#pragma unroll
        for (int e = 0; e < VEC; ++e) pv.v[e] = caxpy_r(rv.v[e], alpha, pv.v[e]);
        st_pack<false>(p + i, pv);
    }
}

template <typename E, int VEC>
__global__ void __launch_bounds__(kThreads) k_cgm_pupdate(SolveState* st) {
    if (st->res.done || st->res.n_iter == 0) return;
    cgm_pupdate_fn<E, VEC>(st->h, st->rc, blockIdx.x, gridDim.x);
}

// A4: one CTA.  P = <p,Ap>; beta = -R0/P; zeta_new_k, beta_k for active shifts.
__device__ __forceinline__ void cgm_scal1_fn(const SolveHeader& h, SolveResult& res, Recur& rc, double P) {
    __shared__ int bad;
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    const double R0 = rc.R1;
    const double beta = -R0 / P;
    const double alpha = rc.alpha.re, beta_prev = rc.beta_prev.re;
    const int na = res.nactive;
    if (!(P > 0.0) || !isfinite(P) || !isfinite(beta)) bad = 1;   // same value from every thread
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = rc.active[a];
        const double z = rc.zeta[k].re, zp = rc.zeta_prev[k].re;
        const double den = beta * alpha * (zp - z) + zp * beta_prev * (1.0 - h.sigma[k] * beta);
        const double zn = z * zp * beta_prev / den;
        const double bk = beta * zn / z;
        if (den == 0.0 || !isfinite(zn) || !isfinite(bk)) bad = 1;
        rc.zeta_new[k].re = zn;
        rc.beta_k[k].re = bk;
        rc.coef[3 * a + 0] = z;                 // zeta_k of this iteration: the lagged p_k update
        rc.coef[3 * a + 1] = rc.alpha_k[k].re;  // alpha_k from the previous scal2
        rc.coef[3 * a + 2] = bk;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        rc.R0 = R0;
        rc.beta.re = beta;
        if (bad) { res.status = MSOLVE_BREAKDOWN; res.done = 1; }
    }
    __syncthreads();
}


// A5: the fused multishift update.  UNR shifts are in flight per thread (2*UNR independent
// 16-byte loads) on top of r and Ap; x_k / p_k are streamed with evict-first hints.  Returns the thread's |r|^2 share.
// STREAM: x_k / p_k with evict-first hints (working sets far beyond L2: every byte is touched once per iteration);
// the whole-solve kernel for systems around the size of L2 passes false so that the vectors stay there.
template <typename E, int VEC, int UNR, bool STREAM = true>
__device__ __forceinline__ double cgm_update_fn(const SolveHeader& h, const SolveResult& res, const Recur& rc, int cta, int ncta) {
    typedef E C;
    typedef typename RealOf<E>::type T;
    typedef Pack<E, VEC> P;
    __shared__ T s_zeta[kMaxShifts], s_alpha[kMaxShifts], s_beta[kMaxShifts];
    __shared__ int s_k[kMaxShifts];
    const int na = res.nactive;
    const bool first = res.n_iter == 0;
    __syncthreads();                              // the arrays may still be read by a previous call (fused kernel)
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        s_k[a] = rc.active[a];
        s_zeta[a] = (T)rc.coef[3 * a + 0];
        s_alpha[a] = (T)rc.coef[3 * a + 1];
        s_beta[a] = (T)rc.coef[3 * a + 2];
    }
    const T beta = (T)rc.beta.re;
    __syncthreads();
    const long long n = h.n, nvec = n / VEC, pks = h.pk_stride, xs = h.x_stride;
    P* r = (P*)h.r;
    const P* q = (const P*)h.q;
    C* x = (C*)h.x;
    C* pk = (C*)h.pk;
    double acc = 0.0;
    const long long stride = (long long)ncta * blockDim.x;
    for (long long i = (long long)cta * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        P rv = ld_pack<false>(r + i);
        const P qv = ld_pack<false>(q + i);
        for (int a0 = 0; a0 < na; a0 += UNR) {
            P xv[UNR], pv[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                if (a0 + u < na && !first) {
                    const int k = s_k[a0 + u];
                    xv[u] = ld_pack<STREAM>((const P*)(x + k * xs) + i);
                    pv[u] = ld_pack<STREAM>((const P*)(pk + k * pks) + i);
                }
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                if (a0 + u < na) {
                    const int k = s_k[a0 + u];
                    const T zk = s_zeta[a0 + u], ak = s_alpha[a0 + u], bk = s_beta[a0 + u];
                    P xo, po;
#pragma unroll
                    for (int e = 0; e < VEC; ++e) {
                        C pe, xe;
                        if (first) { pe = rv.v[e]; xe = cmake<C>(0.0, 0.0); }        // p_k = b, x_k = 0
                        else {
                            pe = clin_r(zk, rv.v[e], ak, pv[u].v[e]);                // l.29 (lagged)
                            xe = xv[u].v[e];
                        }
                        xo.v[e] = caxpy_r(xe, -bk, pe);                              // l.28
                        po.v[e] = pe;
                    }
                    st_pack<STREAM>((P*)(x + k * xs) + i, xo);
                    st_pack<STREAM>((P*)(pk + k * pks) + i, po);
                }
            }
        }
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            rv.v[e] = caxpy_r(rv.v[e], beta, qv.v[e]);                               // l.21
            acc += cnorm2(rv.v[e]);                                                  // l.24
        }
        st_pack<false>(r + i, rv);
    }
    return acc;
}

template <typename E, int VEC, int UNR>
__global__ void __launch_bounds__(kThreads) k_cgm_update(SolveState* st) {
    if (st->res.done) return;
    double acc[1] = {cgm_update_fn<E, VEC, UNR>(st->h, st->res, st->rc, blockIdx.x, gridDim.x)};
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) {
        st->partial[blockIdx.x] = acc[0];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

// ----------------------------------------------------------------------------- CG-M, deferred multishift update
// Alg. 1 l.28-29 touch every x_k and p_k in every iteration: 4 S + 3 vector passes, 2/3 of the
// bytes of an iteration at S = 16.  But p_k(n) = zeta_k(n) r_n + alpha_k(n) p_k(n-1) and x_k(n+1) = x_k(n) -
// beta_k(n) p_k(n) are LINEAR in the residuals with scalar coefficients the recurrences already produce, so over a
// chunk of M iterations that starts with P_k = p_k(n0 - 1), X_k = x_k(n0) in memory
//     p_k(n0 + m - 1) = Ap_k P_k + sum_j Cp_k[j] r_{n0+j},     x_k(n0 + m) = X_k + Ax_k P_k + sum_j Cx_k[j] r_{n0+j}
// where appending iteration n (coefficients zeta, alpha_k, beta_k of cgm_scal1_fn) is
//     Cp_k[j] <- alpha_k Cp_k[j] (j < f),  Cp_k[f] <- zeta,  Ap_k <- alpha_k Ap_k,  Cx_k[j] -= beta_k Cp_k[j],  Ax_k -= beta_k Ap_k.
// The iteration keeps the residuals of the chunk (r lives in a ring of M + 1 vectors, so keeping them costs no
// copy), the scalar kernel keeps the 2 M + 2 coefficients per shift in fp64, and ONE pass per chunk (k_cgm_flush)
// forms p_k and x_k: (M + 4 S) / M vector passes per iteration instead of 4 S; a solve that ends inside its first
// chunk writes every x_k exactly once and never touches p_k.  Scalars, residuals and stopping decisions are those
// of the step-by-step form (they do not depend on x_k, p_k); x_k differs by the order of the additions.
// A shift that stops inside a chunk keeps its coefficients until the flush (the flush walks the shifts that were
// active when the chunk began).
__device__ __forceinline__ void defer_init(Defer& df) {
    if (threadIdx.x == 0) { df.fill = 0; df.s0 = 0; df.first = 1; df.need_begin = 1; df.nlist = 0; df.ticket = 0u; df.r_next = nullptr; }
    __syncthreads();
}

// one CTA, right after cgm_scal1_fn of iteration n: start a chunk if the last one was flushed, append iteration n
__device__ __forceinline__ void cgm_defer_coef_fn(const SolveHeader& h, const SolveResult& res, const Recur& rc, Defer& df) {
    if (res.done) return;                                  // breakdown in this iteration: it is not applied
    const int na = res.nactive;
    if (df.need_begin) {
        for (int a = threadIdx.x; a < na; a += blockDim.x) {
            const int k = rc.active[a];
            df.list[a] = k; df.pos[k] = a; df.Ap[a] = 1.0; df.Ax[a] = 0.0;
            for (int j = 0; j < kDeferMax; ++j) { df.Cp[a * kDeferMax + j] = 0.0; df.Cx[a * kDeferMax + j] = 0.0; }
        }
        __syncthreads();
        if (threadIdx.x == 0) { df.nlist = na; df.need_begin = 0; }
        __syncthreads();
    }
    const int f = df.fill;
    for (int idx = threadIdx.x; idx < na * (f + 1); idx += blockDim.x) {
        const int a = idx / (f + 1), j = idx - a * (f + 1);
        const int la = df.pos[rc.active[a]];
        const double z = rc.coef[3 * a + 0], ak = rc.coef[3 * a + 1], bk = rc.coef[3 * a + 2];
        const double cp = j < f ? ak * df.Cp[la * kDeferMax + j] : z;
        df.Cp[la * kDeferMax + j] = cp;
        df.Cx[la * kDeferMax + j] -= bk * cp;
        if (j == 0) {
            const double ap = ak * df.Ap[la];
            df.Ap[la] = ap;
            df.Ax[la] -= bk * ap;
        }
    }
    if (threadIdx.x == 0) {
        const int slots = h.defer + 1;
        df.r_next = (char*)h.ring + (long long)((df.s0 + f + 1) % slots) * h.ring_stride;
    }
    __syncthreads();
}

// one CTA, right after cgm_scal2_fn: iteration n is complete, r_{n+1} is the residual from here on
__device__ __forceinline__ void cgm_defer_advance(SolveHeader& h, Defer& df) {
    if (threadIdx.x == 0) { df.fill += 1; h.r = df.r_next; }
    __syncthreads();
}

// l.21, 24 alone: r_{n+1} = r_n + beta q into the next slot of the ring; returns the thread's |r_{n+1}|^2 share
template <typename E, int VEC>
__device__ __forceinline__ double cgm_rupdate_fn(const SolveHeader& h, const Recur& rc, const Defer& df, int cta, int ncta) {
    typedef typename RealOf<E>::type T;
    typedef Pack<E, VEC> P;
    const long long nvec = h.n / VEC;
    const P* r = (const P*)h.r;
    const P* q = (const P*)h.q;
    P* rn = (P*)df.r_next;
    const T beta = (T)rc.beta.re;
    const long long stride = (long long)ncta * blockDim.x;
    constexpr int U = kPupdUnroll;
    double acc = 0.0;
    long long i = (long long)cta * blockDim.x + threadIdx.x;
    for (; i + (U - 1) * stride < nvec; i += U * stride) {
        P rv[U], qv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { rv[u] = ld_pack<false>(r + i + u * stride); qv[u] = ld_pack<false>(q + i + u * stride); }
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int e = 0; e < VEC; ++e) { rv[u].v[e] = caxpy_r(rv[u].v[e], beta, qv[u].v[e]); acc += cnorm2(rv[u].v[e]); }
            st_pack<false>(rn + i + u * stride, rv[u]);
        }
    }
    for (; i < nvec; i += stride) {
        P rv = ld_pack<false>(r + i);
        const P qv = ld_pack<false>(q + i);
#pragma unroll
        for (int e = 0; e < VEC; ++e) { rv.v[e] = caxpy_r(rv.v[e], beta, qv.v[e]); acc += cnorm2(rv.v[e]); }
        st_pack<false>(rn + i, rv);
    }
    return acc;
}

template <typename E, int VEC>
__global__ void __launch_bounds__(kThreads) k_cgm_rupdate(SolveState* st) {
    if (st->res.done) return;
    double acc[1] = {cgm_rupdate_fn<E, VEC>(st->h, st->rc, st->df, blockIdx.x, gridDim.x)};
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) {
        st->partial[blockIdx.x] = acc[0];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

// The pass that forms p_k and x_k of a chunk.  It sits at the end of the loop body and does something when the chunk
// is full or the solve has just ended with residuals pending; the last CTA to finish retires the chunk.
// Per element: the chunk's residuals into registers once, then per shift of the chunk's list two loads (unless this
// is the first flush of the solve), 2 cnt multiply-adds per component, and the stores (p_k only while the shift is
// still iterating).  Coefficients are rounded to the element's precision, sums run in it, as in cgm_update_fn.
template <typename E, int VEC, int UNR>
__global__ void __launch_bounds__(kThreads) k_cgm_flush(SolveState* st) {
    typedef E C;
    typedef typename RealOf<E>::type T;
    typedef Pack<E, VEC> P;
    const SolveHeader& h = st->h;
    Defer& df = st->df;
    const int cnt = df.fill;
    const bool ended = st->res.done != 0;
    if (!(cnt == h.defer || (ended && cnt > 0))) return;            // the same decision in every CTA
    extern __shared__ __align__(16) unsigned char flush_dyn[];            // 2 x kMaxShifts x kDeferMax coefficients: beyond 48 KB in fp64
    T* s_cp = (T*)flush_dyn;
    T* s_cx = s_cp + kMaxShifts * kDeferMax;
    __shared__ T s_ap[kMaxShifts], s_ax[kMaxShifts];
    __shared__ int s_k[kMaxShifts], s_wp[kMaxShifts];
    __shared__ const P* s_r[kDeferMax];
    __shared__ unsigned int s_last;
    const int nl = df.nlist;
    const bool first = df.first != 0;
    for (int a = threadIdx.x; a < nl; a += blockDim.x) {
        const int k = df.list[a];
        s_k[a] = k;
        s_wp[a] = !ended && st->res.conv_iter[k] < 0;              // p_k is needed again
        s_ap[a] = (T)df.Ap[a]; s_ax[a] = (T)df.Ax[a];
    }
    for (int idx = threadIdx.x; idx < nl * cnt; idx += blockDim.x) {
        const int a = idx / cnt, j = idx - a * cnt;
        s_cp[a * kDeferMax + j] = (T)df.Cp[a * kDeferMax + j];
        s_cx[a * kDeferMax + j] = (T)df.Cx[a * kDeferMax + j];
    }
    if (threadIdx.x < cnt) s_r[threadIdx.x] = (const P*)((const char*)h.ring + (long long)((df.s0 + threadIdx.x) % (h.defer + 1)) * h.ring_stride);
    __syncthreads();
    const long long nvec = h.n / VEC, pks = h.pk_stride, xs = h.x_stride;
    C* x = (C*)h.x;
    C* pk = (C*)h.pk;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        P rj[kDeferMax];
#pragma unroll
        for (int j = 0; j < kDeferMax; ++j)
            if (j < cnt) rj[j] = ld_pack<true>(s_r[j] + i);
        for (int a0 = 0; a0 < nl; a0 += UNR) {
            P xv[UNR], pv[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                if (a0 + u < nl && !first) {
                    const int k = s_k[a0 + u];
                    xv[u] = ld_pack<true>((const P*)(x + k * xs) + i);
                    pv[u] = ld_pack<true>((const P*)(pk + k * pks) + i);
                }
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                if (a0 + u < nl) {
                    const int a = a0 + u, k = s_k[a];
                    const T* cx = s_cx + a * kDeferMax;
                    P xo;
#pragma unroll
                    for (int e = 0; e < VEC; ++e)
                        xo.v[e] = first ? cmake<C>(0.0, 0.0) : caxpy_r(xv[u].v[e], s_ax[a], pv[u].v[e]);
#pragma unroll
                    for (int j = 0; j < kDeferMax; ++j) {
                        if (j < cnt) {
#pragma unroll
                            for (int e = 0; e < VEC; ++e) xo.v[e] = caxpy_r(xo.v[e], cx[j], rj[j].v[e]);
                        }
                    }
                    st_pack<true>((P*)(x + k * xs) + i, xo);
                    if (s_wp[a]) {                           // p_k only while it is needed again (half of the multiply-adds)
                        const T* cp = s_cp + a * kDeferMax;
                        P po;
#pragma unroll
                        for (int e = 0; e < VEC; ++e)
                            po.v[e] = first ? cmake<C>(0.0, 0.0) : caxpy_r(cmake<C>(0.0, 0.0), s_ap[a], pv[u].v[e]);
#pragma unroll
                        for (int j = 0; j < kDeferMax; ++j) {
                            if (j < cnt) {
#pragma unroll
                                for (int e = 0; e < VEC; ++e) po.v[e] = caxpy_r(po.v[e], cp[j], rj[j].v[e]);
                            }
                        }
                        st_pack<true>((P*)(pk + k * pks) + i, po);
                    }
                }
            }
        }
    }
    // the last CTA to get here retires the chunk: the next one starts at the current residual
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&df.ticket, 1u) == gridDim.x - 1 ? 1u : 0u;
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        df.s0 = (df.s0 + cnt) % (h.defer + 1);
        df.fill = 0; df.first = 0; df.need_begin = 1; df.ticket = 0u;
        __threadfence();
    }
}

// Loop control shared by both algorithms: called by thread 0 after the per-shift stop test.
__device__ __forceinline__ void finish_iteration(const SolveHeader& h, SolveResult& res, Recur& rc, bool bad) {
    // compact the active list in order (S <= 128: serial is fine)
    const int na = res.nactive;
    int m = 0;
    for (int a = 0; a < na; ++a) {
        const int k = rc.active[a];
        if (res.conv_iter[k] < 0) rc.active[m++] = k;
    }
    res.nactive = m;
    if (bad) { res.status = MSOLVE_BREAKDOWN; res.done = 1; }
    else if (m == 0) { res.status = MSOLVE_OK; res.done = 1; }
    else if (res.n_iter >= h.max_iter) { res.status = MSOLVE_MAXITER; res.done = 1; }
}

// A6: one CTA.  R1 -> alpha, alpha_k; zeta shuffle; per-shift stop test; loop control.  `hist` = the history
// buffer or NULL (in the fused kernel only CTA 0 passes it).
__device__ __forceinline__ void cgm_scal2_fn(const SolveHeader& h, SolveResult& res, Recur& rc, const double* rhs_norm,
                                             double R1, double* hist) {
    const double R0 = rc.R0;
    const double alpha_next = R1 / R0;
    const int na = res.nactive;
    const int it = res.n_iter + 1;
    const double rnorm = sqrt(R1), bnorm = rc.bnorm, tol = h.tol;
    const bool force = h.force_all != 0, base_rule = h.stop_rule == 1, psn = h.per_shift_norm != 0;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = rc.active[a];
        const double zn = rc.zeta_new[k].re, z = rc.zeta[k].re;
        const double ratio = zn / z;
        rc.alpha_k[k].re = alpha_next * ratio * ratio;                  // l.26
        rc.zeta_prev[k].re = z;                                         // l.30
        rc.zeta[k].re = zn;                                             // l.31
        const double nk = psn ? rhs_norm[k] : bnorm;                    // eq. (6): relative to the shift's own ||b_k||
        const double rel = fabs(zn) * rnorm / nk;
        res.relres[k] = rel;
        // l.15: per shift (R15), or literally on the unshifted residual (stop_rule = 1)
        if (!force && (base_rule ? rnorm : fabs(zn) * rnorm) <= tol * nk) res.conv_iter[k] = it;
    }
    __syncthreads();
    // msolve_set_history: row it-1 = beta, alpha_next, R1, then zeta_new[S], beta_k[S], alpha_k[S] (frozen shifts
    // keep the values of their last active iteration)
    if (hist && it <= h.hist_cap) {
        const int S = h.S;
        double* hr = hist + (size_t)(it - 1) * (size_t)(3 + 3 * S);
        if (threadIdx.x == 0) { hr[0] = rc.beta.re; hr[1] = alpha_next; hr[2] = R1; }
        for (int k = threadIdx.x; k < S; k += blockDim.x) {
            hr[3 + k] = rc.zeta_new[k].re; hr[3 + S + k] = rc.beta_k[k].re; hr[3 + 2 * S + k] = rc.alpha_k[k].re;
        }
    }
    if (threadIdx.x == 0) {
        rc.R1 = R1;
        rc.beta_prev.re = rc.beta.re;                                   // l.17
        rc.alpha.re = alpha_next;                                       // l.25
        res.n_iter = it;                                                // l.32
        finish_iteration(h, res, rc, !isfinite(R1) || !isfinite(alpha_next));
    }
    __syncthreads();
}


// ----------------------------------------------------------------------------- BiCGStab-M
// after SpMV#1: beta = -delta/<r0,q>; zeta_new_k, beta_k (complex).
__device__ __forceinline__ void bi_scal1_fn(const SolveHeader& h, SolveResult& res, Recur& rc, zd r0q) {
    __shared__ int bad;
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    const zd delta = rc.delta;
    const zd beta = zneg(zdiv(delta, r0q));
    const zd alpha = rc.alpha, beta_prev = rc.beta_prev;
    if (zzero(r0q) || zzero(delta) || !zfinite(r0q) || !zfinite(beta)) bad = 1;
    const int na = res.nactive;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = rc.active[a];
        const zd z = rc.zeta[k], zp = rc.zeta_prev[k];
        const zd one_sb = {1.0 - h.sigma[k] * beta.re, -h.sigma[k] * beta.im};
        const zd den = zadd(zmul(zmul(beta, alpha), zsub(zp, z)), zmul(zmul(zp, beta_prev), one_sb));
        const zd zn = zdiv(zmul(zmul(z, zp), beta_prev), den);
        const zd bk = zdiv(zmul(beta, zn), z);
        if (zzero(den) || !zfinite(zn) || !zfinite(bk)) bad = 1;
        rc.zeta_new[k] = zn;
        rc.beta_k[k] = bk;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        rc.beta = beta;
        if (bad) { res.status = MSOLVE_BREAKDOWN; res.done = 1; }
    }
    __syncthreads();
}


// s <- r + beta q
template <typename E, int VEC>
__device__ __forceinline__ void bi_supdate_fn(const SolveHeader& h, const Recur& rc, int cta, int ncta) {
    typedef E C;
    typedef Pack<E, VEC> P;
    const long long nvec = h.n / VEC;
    const P* r = (const P*)h.r;
    const P* q = (const P*)h.q;
    P* s = (P*)h.s;
    const C beta = cmake<C>(rc.beta.re, rc.beta.im);
    const long long stride = (long long)ncta * blockDim.x;
    for (long long i = (long long)cta * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const P rv = ld_pack<false>(r + i), qv = ld_pack<false>(q + i);
        P sv;
#pragma unroll
        for (int e = 0; e < VEC; ++e) sv.v[e] = cfma(beta, qv.v[e], rv.v[e]);
        st_pack<false>(s + i, sv);
    }
}

template <typename E, int VEC>
__global__ void __launch_bounds__(kThreads) k_bi_supdate(SolveState* st) {
    if (st->res.done) return;
    bi_supdate_fn<E, VEC>(st->h, st->rc, blockIdx.x, gridDim.x);
}

// after SpMV#2: chi, chi_k, rho'_k, delta' = -chi <r0,t>, alpha' = -beta delta'/(delta chi), alpha_k;
// writes the 7 complex coefficients per active shift used by the fused update.  s5 = <t,s> (2), <t,t>, <r0,t> (2).
__device__ __forceinline__ void bi_scal2_fn(const SolveHeader& h, SolveResult& res, Recur& rc, const double* s5) {
    __shared__ int bad;
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    const zd ts = {s5[0], s5[1]};
    const double tt = s5[2];
    const zd r0t = {s5[3], s5[4]};
    const zd chi = {ts.re / tt, ts.im / tt};
    const zd beta = rc.beta, delta = rc.delta;
    const zd delta_new = zneg(zmul(chi, r0t));               // <r0, s - chi t> with <r0,s> = 0
    const zd alpha_new = zneg(zdiv(zmul(beta, delta_new), zmul(delta, chi)));
    if (!(tt > 0.0) || !isfinite(tt) || !zfinite(ts) || zzero(chi) || !zfinite(alpha_new)) bad = 1;
    const int na = res.nactive;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = rc.active[a];
        const double sg = h.sigma[k];
        const zd one_cs = {1.0 + chi.re * sg, chi.im * sg};
        if (zzero(one_cs)) bad = 1;
        const zd chik = zdiv(chi, one_cs);
        const zd rho = rc.rho[k];
        const zd rho_new = zdiv(rho, one_cs);
        const zd zn = rc.zeta_new[k], z = rc.zeta[k], bk = rc.beta_k[k];
        const zd ratio = zdiv(zn, z);
        const zd ak = zmul(alpha_new, zmul(ratio, ratio));
        rc.chi_k[k] = chik;
        rc.rho_new[k] = rho_new;
        rc.alpha_k[k] = ak;
        const zd cs = zmul(zmul(chik, rho), zn);             // x_k += cs * s
        const zd zr = zmul(zn, rho_new);                     // p_k = zr * r' + ...
        const zd cb = zdiv(chik, bk);
        const zd zs = zmul(zn, rho);                         // s^sigma = zs * s
        const zd zo = zmul(z, rho);                          // r^sigma = zo * r
        if (!zfinite(cs) || !zfinite(zr) || !zfinite(cb) || !zfinite(ak)) bad = 1;
        double* c = rc.coef + 14 * a;
        c[0] = bk.re; c[1] = bk.im; c[2] = cs.re; c[3] = cs.im; c[4] = zr.re; c[5] = zr.im;
        c[6] = ak.re; c[7] = ak.im; c[8] = cb.re; c[9] = cb.im; c[10] = zs.re; c[11] = zs.im;
        c[12] = zo.re; c[13] = zo.im;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        rc.chi = chi;
        rc.delta_new = delta_new;
        rc.alpha_new = alpha_new;
        if (bad) { res.status = MSOLVE_BREAKDOWN; res.done = 1; }
    }
    __syncthreads();
}


// The fused BiCGStab-M update: per element read r, s, t, q, p once;
//   r' = s - chi t ; p <- r' + alpha'(p - chi q) ; |r'|^2 partials; per active shift
//   x_k <- (x_k - beta_k p_k) + cs_k s ; p_k <- zr_k r' + alpha_k ( p_k - cb_k ( zs_k s - zo_k r ) ).
template <typename E, int VEC, int UNR, bool STREAM = true>
__device__ __forceinline__ double bi_update_fn(const SolveHeader& h, const SolveResult& res, const Recur& rc, int cta, int ncta) {
    typedef E C;
    typedef Pack<E, VEC> P;
    __shared__ C s_c[kMaxShifts * 7];
    __shared__ int s_k[kMaxShifts];
    const int na = res.nactive;
    const bool first = res.n_iter == 0;
    __syncthreads();
    for (int a = threadIdx.x; a < na; a += blockDim.x) s_k[a] = rc.active[a];
    for (int j = threadIdx.x; j < 7 * na; j += blockDim.x) s_c[j] = cmake<C>(rc.coef[2 * j], rc.coef[2 * j + 1]);
    const C chi = cmake<C>(rc.chi.re, rc.chi.im);
    const C alpha_new = cmake<C>(rc.alpha_new.re, rc.alpha_new.im);
    __syncthreads();
    const long long n = h.n, nvec = n / VEC, pks = h.pk_stride, xs = h.x_stride;
    P* r = (P*)h.r;
    P* p = (P*)h.p;
    const P* s = (const P*)h.s;
    const P* t = (const P*)h.t;
    const P* q = (const P*)h.q;
    C* x = (C*)h.x;
    C* pk = (C*)h.pk;
    double acc = 0.0;
    const long long stride = (long long)ncta * blockDim.x;
    for (long long i = (long long)cta * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const P rv = ld_pack<false>(r + i), sv = ld_pack<false>(s + i), tv = ld_pack<false>(t + i);
        const P qv = ld_pack<false>(q + i);
        P pv0 = ld_pack<false>(p + i);
        P rn;
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            rn.v[e] = csub(sv.v[e], cmul(chi, tv.v[e]));
            pv0.v[e] = cadd(rn.v[e], cmul(alpha_new, csub(pv0.v[e], cmul(chi, qv.v[e]))));
            acc += cnorm2(rn.v[e]);
        }
        for (int a0 = 0; a0 < na; a0 += UNR) {
            P xv[UNR], pv[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                if (a0 + u < na && !first) {
                    const int k = s_k[a0 + u];
                    xv[u] = ld_pack<STREAM>((const P*)(x + k * xs) + i);
                    pv[u] = ld_pack<STREAM>((const P*)(pk + k * pks) + i);
                }
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                if (a0 + u < na) {
                    const int k = s_k[a0 + u];
                    const C* c = s_c + 7 * (a0 + u);
                    P xo, po;
#pragma unroll
                    for (int e = 0; e < VEC; ++e) {
                        const C pe = first ? rv.v[e] : pv[u].v[e];                   // p_k = b = r at n = 0
                        const C xe = first ? cmake<C>(0.0, 0.0) : xv[u].v[e];
                        xo.v[e] = cadd(csub(xe, cmul(c[0], pe)), cmul(c[1], sv.v[e]));
                        const C ds = csub(cmul(c[5], sv.v[e]), cmul(c[6], rv.v[e]));
                        po.v[e] = cadd(cmul(c[2], rn.v[e]), cmul(c[3], csub(pe, cmul(c[4], ds))));
                    }
                    st_pack<STREAM>((P*)(x + k * xs) + i, xo);
                    st_pack<STREAM>((P*)(pk + k * pks) + i, po);
                }
            }
        }
        st_pack<false>(r + i, rn);
        st_pack<false>(p + i, pv0);
    }
    return acc;
}

template <typename E, int VEC, int UNR>
__global__ void __launch_bounds__(kThreads) k_bi_update(SolveState* st) {
    if (st->res.done) return;
    double acc[1] = {bi_update_fn<E, VEC, UNR>(st->h, st->res, st->rc, blockIdx.x, gridDim.x)};
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) {
        st->partial[blockIdx.x] = acc[0];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

// end of iteration: |r'|^2 -> shuffle zeta/rho/delta/alpha/beta, per-shift stop test, loop control.
__device__ __forceinline__ void bi_scal3_fn(const SolveHeader& h, SolveResult& res, Recur& rc, const double* rhs_norm,
                                            double rr, double* hist) {
    const int na = res.nactive;
    const int it = res.n_iter + 1;
    const double rnorm = sqrt(rr), bnorm = rc.bnorm, tol = h.tol;
    const bool force = h.force_all != 0, base_rule = h.stop_rule == 1, psn = h.per_shift_norm != 0;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = rc.active[a];
        const zd zn = rc.zeta_new[k], rn = rc.rho_new[k];
        rc.zeta_prev[k] = rc.zeta[k];
        rc.zeta[k] = zn;
        rc.rho[k] = rn;
        const double zr = zabs(zmul(zn, rn));
        const double nk = psn ? rhs_norm[k] : bnorm;
        res.relres[k] = zr * rnorm / nk;
        if (!force && (base_rule ? rnorm : zr * rnorm) <= tol * nk) res.conv_iter[k] = it;
    }
    __syncthreads();
    // msolve_set_history: row it-1 = beta, chi, alpha' (complex), |r'|^2, 0, then zeta_new[S], beta_k[S], chi_k[S] (complex)
    if (hist && it <= h.hist_cap) {
        const int S = h.S;
        double* hr = hist + (size_t)(it - 1) * (size_t)(8 + 6 * S);
        if (threadIdx.x == 0) {
            hr[0] = rc.beta.re; hr[1] = rc.beta.im; hr[2] = rc.chi.re; hr[3] = rc.chi.im;
            hr[4] = rc.alpha_new.re; hr[5] = rc.alpha_new.im; hr[6] = rr; hr[7] = 0.0;
        }
        for (int k = threadIdx.x; k < S; k += blockDim.x) {
            hr[8 + 2 * k] = rc.zeta_new[k].re; hr[8 + 2 * k + 1] = rc.zeta_new[k].im;
            hr[8 + 2 * S + 2 * k] = rc.beta_k[k].re; hr[8 + 2 * S + 2 * k + 1] = rc.beta_k[k].im;
            hr[8 + 4 * S + 2 * k] = rc.chi_k[k].re; hr[8 + 4 * S + 2 * k + 1] = rc.chi_k[k].im;
        }
    }
    if (threadIdx.x == 0) {
        rc.R1 = rr;
        rc.delta = rc.delta_new;
        rc.alpha = rc.alpha_new;
        rc.beta_prev = rc.beta;
        res.n_iter = it;
        finish_iteration(h, res, rc, !isfinite(rr));
    }
    __syncthreads();
}


}  // namespace msolve
