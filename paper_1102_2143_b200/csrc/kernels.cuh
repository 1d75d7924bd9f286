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
__global__ void __launch_bounds__(kThreads) k_init_vectors(SolveState* st) {
    typedef Pack<E, VEC> P;
    const long long nvec = st->h.n / VEC;
    const P* b = (const P*)st->h.b;
    P* r = (P*)st->h.r;
    P* p = (P*)st->h.p;
    double acc[1] = {0.0};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const P bv = ld_pack<false>(b + i);
        st_pack<false>(r + i, bv);
        st_pack<false>(p + i, bv);
#pragma unroll
        for (int e = 0; e < VEC; ++e) acc[0] += cnorm2(bv.v[e]);
    }
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) {
        st->partial[blockIdx.x] = acc[0];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

// Scalars of l.2-8, 13-14 and the BiCGStab-M analogue; b = 0 ends the solve at once.
__global__ void __launch_bounds__(kThreads) k_init_state(SolveState* st) {
    __shared__ double red[32];
    double s[1];
    reduce_partials<1>(st, s, red);
    const int S = st->h.S;
    for (int k = threadIdx.x; k < S; k += blockDim.x) {
        st->zeta_prev[k] = {1.0, 0.0}; st->zeta[k] = {1.0, 0.0}; st->zeta_new[k] = {1.0, 0.0};
        st->rho[k] = {1.0, 0.0}; st->rho_new[k] = {1.0, 0.0};
        st->beta_k[k] = {0.0, 0.0}; st->alpha_k[k] = {0.0, 0.0}; st->chi_k[k] = {0.0, 0.0};
        st->active[k] = k;
        st->res.conv_iter[k] = (s[0] == 0.0) ? 0 : -1;
        st->res.relres[k] = (s[0] == 0.0) ? 0.0 : 1.0;
    }
    if (threadIdx.x == 0) {
        st->alpha = {0.0, 0.0}; st->beta = {0.0, 0.0}; st->beta_prev = {1.0, 0.0};
        st->delta = {s[0], 0.0};            // <r0,r> = <b,b>
        st->chi = {0.0, 0.0}; st->alpha_new = {0.0, 0.0}; st->delta_new = {0.0, 0.0};
        st->R0 = s[0]; st->R1 = s[0]; st->bnorm = sqrt(s[0]);
        st->res.n_iter = 0;
        st->res.status = MSOLVE_OK;
        st->res.nactive = S;
        st->res.zero_rhs = (s[0] == 0.0);
        st->res.done = (s[0] == 0.0) || !isfinite(s[0]) || st->h.max_iter <= 0;
        if (!isfinite(s[0])) st->res.status = MSOLVE_BREAKDOWN;
        else if (s[0] != 0.0 && st->h.max_iter <= 0) st->res.status = MSOLVE_MAXITER;
    }
}

constexpr int kPupdUnroll = 4;   // 2 * 4 independent 16-byte loads in flight per thread
// ----------------------------------------------------------------------------- CG-M
// A1: p <- r + alpha p  (l.27; at n = 0 p = b already)
template <typename E, int VEC>
__global__ void __launch_bounds__(kThreads) k_cgm_pupdate(SolveState* st) {
    if (st->res.done || st->res.n_iter == 0) return;
    typedef typename RealOf<E>::type T;
    typedef Pack<E, VEC> P;
    const long long nvec = st->h.n / VEC;
    const P* r = (const P*)st->h.r;
    P* p = (P*)st->h.p;
    const T alpha = (T)st->alpha.re;
    const long long stride = (long long)gridDim.x * blockDim.x;
    constexpr int U = kPupdUnroll;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
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

// A4: one CTA.  P = sum of partials; beta = -R0/P; zeta_new_k, beta_k for active shifts.
__global__ void __launch_bounds__(kThreads) k_cgm_scal1(SolveState* st) {
    if (st->res.done) return;
    __shared__ double red[32];
    __shared__ int bad;
    double s[1];
    if (threadIdx.x == 0) bad = 0;
    reduce_partials<1>(st, s, red);
    const double P = s[0];
    const double R0 = st->R1;
    const double beta = -R0 / P;
    const double alpha = st->alpha.re, beta_prev = st->beta_prev.re;
    const int na = st->res.nactive;
    if (!(P > 0.0) || !isfinite(P) || !isfinite(beta)) bad = 1;   // same value from every thread
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = st->active[a];
        const double z = st->zeta[k].re, zp = st->zeta_prev[k].re;
        const double den = beta * alpha * (zp - z) + zp * beta_prev * (1.0 - st->h.sigma[k] * beta);
        const double zn = z * zp * beta_prev / den;
        const double bk = beta * zn / z;
        if (den == 0.0 || !isfinite(zn) || !isfinite(bk)) bad = 1;
        st->zeta_new[k].re = zn;
        st->beta_k[k].re = bk;
        st->coef[3 * a + 0] = z;                 // zeta_k of this iteration: the lagged p_k update
        st->coef[3 * a + 1] = st->alpha_k[k].re; // alpha_k from the previous scal2
        st->coef[3 * a + 2] = bk;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st->R0 = R0;
        st->beta.re = beta;
        if (bad) { st->res.status = MSOLVE_BREAKDOWN; st->res.done = 1; }
    }
}

// A5: the fused multishift update.  UNR shifts are in flight per thread (2*UNR independent
// 16-byte loads) on top of r and Ap; x_k / p_k are streamed with evict-first hints.
template <typename E, int VEC, int UNR>
__global__ void __launch_bounds__(kThreads) k_cgm_update(SolveState* st) {
    if (st->res.done) return;
    typedef E C;
    typedef typename RealOf<E>::type T;
    typedef Pack<E, VEC> P;
    __shared__ T s_zeta[kMaxShifts], s_alpha[kMaxShifts], s_beta[kMaxShifts];
    __shared__ int s_k[kMaxShifts];
    const int na = st->res.nactive;
    const bool first = st->res.n_iter == 0;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        s_k[a] = st->active[a];
        s_zeta[a] = (T)st->coef[3 * a + 0];
        s_alpha[a] = (T)st->coef[3 * a + 1];
        s_beta[a] = (T)st->coef[3 * a + 2];
    }
    const T beta = (T)st->beta.re;
    __syncthreads();
    const long long n = st->h.n, nvec = n / VEC, pks = st->h.pk_stride;
    P* r = (P*)st->h.r;
    const P* q = (const P*)st->h.q;
    C* x = (C*)st->h.x;
    C* pk = (C*)st->h.pk;
    double acc[1] = {0.0};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        P rv = ld_pack<false>(r + i);
        const P qv = ld_pack<false>(q + i);
        for (int a0 = 0; a0 < na; a0 += UNR) {
            P xv[UNR], pv[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                if (a0 + u < na && !first) {
                    const int k = s_k[a0 + u];
                    xv[u] = ld_pack<true>((const P*)(x + k * n) + i);
                    pv[u] = ld_pack<true>((const P*)(pk + k * pks) + i);
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
                    st_pack<true>((P*)(x + k * n) + i, xo);
                    st_pack<true>((P*)(pk + k * pks) + i, po);
                }
            }
        }
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            rv.v[e] = caxpy_r(rv.v[e], beta, qv.v[e]);                               // l.21
            acc[0] += cnorm2(rv.v[e]);                                               // l.24
        }
        st_pack<false>(r + i, rv);
    }
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) {
        st->partial[blockIdx.x] = acc[0];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

// Loop control shared by both algorithms: called by thread 0 after the per-shift stop test.
__device__ __forceinline__ void finish_iteration(SolveState* st, bool bad) {
    // compact the active list in order (S <= 128: serial is fine)
    const int na = st->res.nactive;
    int m = 0;
    for (int a = 0; a < na; ++a) {
        const int k = st->active[a];
        if (st->res.conv_iter[k] < 0) st->active[m++] = k;
    }
    st->res.nactive = m;
    if (bad) { st->res.status = MSOLVE_BREAKDOWN; st->res.done = 1; }
    else if (m == 0) { st->res.status = MSOLVE_OK; st->res.done = 1; }
    else if (st->res.n_iter >= st->h.max_iter) { st->res.status = MSOLVE_MAXITER; st->res.done = 1; }
}

// A6: one CTA.  R1 -> alpha, alpha_k; zeta shuffle; per-shift stop test; loop control.
// `cond` is the WHILE node's handle (use_cond = 0 in chunked mode).
__global__ void __launch_bounds__(kThreads) k_cgm_scal2(SolveState* st, cudaGraphConditionalHandle cond, int use_cond) {
    if (st->res.done) { if (use_cond && threadIdx.x == 0) cudaGraphSetConditional(cond, 0); return; }
    __shared__ double red[32];
    double s[1];
    reduce_partials<1>(st, s, red);
    const double R1 = s[0], R0 = st->R0;
    const double alpha_next = R1 / R0;
    const int na = st->res.nactive;
    const int it = st->res.n_iter + 1;
    const double rnorm = sqrt(R1), bnorm = st->bnorm, tol = st->h.tol;
    const bool force = st->h.force_all != 0, base_rule = st->h.stop_rule == 1, psn = st->h.per_shift_norm != 0;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = st->active[a];
        const double zn = st->zeta_new[k].re, z = st->zeta[k].re;
        const double ratio = zn / z;
        st->alpha_k[k].re = alpha_next * ratio * ratio;                 // l.26
        st->zeta_prev[k].re = z;                                        // l.30
        st->zeta[k].re = zn;                                            // l.31
        const double nk = psn ? st->rhs_norm[k] : bnorm;               // eq. (6): relative to the shift's own ||b_k||
        const double rel = fabs(zn) * rnorm / nk;
        st->res.relres[k] = rel;
        // l.15: per shift (R15), or literally on the unshifted residual (stop_rule = 1)
        if (!force && (base_rule ? rnorm : fabs(zn) * rnorm) <= tol * nk) st->res.conv_iter[k] = it;
    }
    // msolve_set_history: row it-1 = beta, alpha_next, R1, then zeta_new[S], beta_k[S], alpha_k[S] (frozen shifts
    // keep the values of their last active iteration)
    if (st->h.hist && it <= st->h.hist_cap) {
        __syncthreads();
        const int S = st->h.S;
        double* h = st->h.hist + (size_t)(it - 1) * (size_t)(3 + 3 * S);
        if (threadIdx.x == 0) { h[0] = st->beta.re; h[1] = alpha_next; h[2] = R1; }
        for (int k = threadIdx.x; k < S; k += blockDim.x) {
            h[3 + k] = st->zeta_new[k].re; h[3 + S + k] = st->beta_k[k].re; h[3 + 2 * S + k] = st->alpha_k[k].re;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st->R1 = R1;
        st->beta_prev.re = st->beta.re;                                 // l.17
        st->alpha.re = alpha_next;                                      // l.25
        st->res.n_iter = it;                                            // l.32
        finish_iteration(st, !isfinite(R1) || !isfinite(alpha_next));
        if (use_cond) cudaGraphSetConditional(cond, st->res.done ? 0u : 1u);
    }
}

// ----------------------------------------------------------------------------- BiCGStab-M
// after SpMV#1: beta = -delta/<r0,q>; zeta_new_k, beta_k (complex).
__global__ void __launch_bounds__(kThreads) k_bi_scal1(SolveState* st) {
    if (st->res.done) return;
    __shared__ double red[2 * 32];
    __shared__ int bad;
    double s[2];
    if (threadIdx.x == 0) bad = 0;
    reduce_partials<2>(st, s, red);
    const zd r0q = {s[0], s[1]};
    const zd delta = st->delta;
    const zd beta = zneg(zdiv(delta, r0q));
    const zd alpha = st->alpha, beta_prev = st->beta_prev;
    if (zzero(r0q) || zzero(delta) || !zfinite(r0q) || !zfinite(beta)) bad = 1;
    const int na = st->res.nactive;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = st->active[a];
        const zd z = st->zeta[k], zp = st->zeta_prev[k];
        const zd one_sb = {1.0 - st->h.sigma[k] * beta.re, -st->h.sigma[k] * beta.im};
        const zd den = zadd(zmul(zmul(beta, alpha), zsub(zp, z)), zmul(zmul(zp, beta_prev), one_sb));
        const zd zn = zdiv(zmul(zmul(z, zp), beta_prev), den);
        const zd bk = zdiv(zmul(beta, zn), z);
        if (zzero(den) || !zfinite(zn) || !zfinite(bk)) bad = 1;
        st->zeta_new[k] = zn;
        st->beta_k[k] = bk;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st->beta = beta;
        if (bad) { st->res.status = MSOLVE_BREAKDOWN; st->res.done = 1; }
    }
}

// s <- r + beta q
template <typename E, int VEC>
__global__ void __launch_bounds__(kThreads) k_bi_supdate(SolveState* st) {
    if (st->res.done) return;
    typedef E C;
    typedef Pack<E, VEC> P;
    const long long nvec = st->h.n / VEC;
    const P* r = (const P*)st->h.r;
    const P* q = (const P*)st->h.q;
    P* s = (P*)st->h.s;
    const C beta = cmake<C>(st->beta.re, st->beta.im);
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const P rv = ld_pack<false>(r + i), qv = ld_pack<false>(q + i);
        P sv;
#pragma unroll
        for (int e = 0; e < VEC; ++e) sv.v[e] = cfma(beta, qv.v[e], rv.v[e]);
        st_pack<false>(s + i, sv);
    }
}

// after SpMV#2: chi, chi_k, rho'_k, delta' = -chi <r0,t>, alpha' = -beta delta'/(delta chi), alpha_k;
// writes the 7 complex coefficients per active shift used by k_bi_update.
__global__ void __launch_bounds__(kThreads) k_bi_scal2(SolveState* st) {
    if (st->res.done) return;
    __shared__ double red[5 * 32];
    __shared__ int bad;
    double s[5];
    if (threadIdx.x == 0) bad = 0;
    reduce_partials<5>(st, s, red);
    const zd ts = {s[0], s[1]};
    const double tt = s[2];
    const zd r0t = {s[3], s[4]};
    const zd chi = {ts.re / tt, ts.im / tt};
    const zd beta = st->beta, delta = st->delta;
    const zd delta_new = zneg(zmul(chi, r0t));               // <r0, s - chi t> with <r0,s> = 0
    const zd alpha_new = zneg(zdiv(zmul(beta, delta_new), zmul(delta, chi)));
    if (!(tt > 0.0) || !isfinite(tt) || !zfinite(ts) || zzero(chi) || !zfinite(alpha_new)) bad = 1;
    const int na = st->res.nactive;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = st->active[a];
        const double sg = st->h.sigma[k];
        const zd one_cs = {1.0 + chi.re * sg, chi.im * sg};
        if (zzero(one_cs)) bad = 1;
        const zd chik = zdiv(chi, one_cs);
        const zd rho = st->rho[k];
        const zd rho_new = zdiv(rho, one_cs);
        const zd zn = st->zeta_new[k], z = st->zeta[k], bk = st->beta_k[k];
        const zd ratio = zdiv(zn, z);
        const zd ak = zmul(alpha_new, zmul(ratio, ratio));
        st->chi_k[k] = chik;
        st->rho_new[k] = rho_new;
        st->alpha_k[k] = ak;
        const zd cs = zmul(zmul(chik, rho), zn);             // x_k += cs * s
        const zd zr = zmul(zn, rho_new);                     // p_k = zr * r' + ...
        const zd cb = zdiv(chik, bk);
        const zd zs = zmul(zn, rho);                         // s^sigma = zs * s
        const zd zo = zmul(z, rho);                          // r^sigma = zo * r
        if (!zfinite(cs) || !zfinite(zr) || !zfinite(cb) || !zfinite(ak)) bad = 1;
        double* c = st->coef + 14 * a;
        c[0] = bk.re; c[1] = bk.im; c[2] = cs.re; c[3] = cs.im; c[4] = zr.re; c[5] = zr.im;
        c[6] = ak.re; c[7] = ak.im; c[8] = cb.re; c[9] = cb.im; c[10] = zs.re; c[11] = zs.im;
        c[12] = zo.re; c[13] = zo.im;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st->chi = chi;
        st->delta_new = delta_new;
        st->alpha_new = alpha_new;
        if (bad) { st->res.status = MSOLVE_BREAKDOWN; st->res.done = 1; }
    }
}

// The fused BiCGStab-M update: per element read r, s, t, q, p once;
//   r' = s - chi t ; p <- r' + alpha'(p - chi q) ; |r'|^2 partials; per active shift
//   x_k <- (x_k - beta_k p_k) + cs_k s ; p_k <- zr_k r' + alpha_k ( p_k - cb_k ( zs_k s - zo_k r ) ).
template <typename E, int VEC, int UNR>
__global__ void __launch_bounds__(kThreads) k_bi_update(SolveState* st) {
    if (st->res.done) return;
    typedef E C;
    typedef Pack<E, VEC> P;
    __shared__ C s_c[kMaxShifts * 7];
    __shared__ int s_k[kMaxShifts];
    const int na = st->res.nactive;
    const bool first = st->res.n_iter == 0;
    for (int a = threadIdx.x; a < na; a += blockDim.x) s_k[a] = st->active[a];
    for (int j = threadIdx.x; j < 7 * na; j += blockDim.x) s_c[j] = cmake<C>(st->coef[2 * j], st->coef[2 * j + 1]);
    const C chi = cmake<C>(st->chi.re, st->chi.im);
    const C alpha_new = cmake<C>(st->alpha_new.re, st->alpha_new.im);
    __syncthreads();
    const long long n = st->h.n, nvec = n / VEC, pks = st->h.pk_stride;
    P* r = (P*)st->h.r;
    P* p = (P*)st->h.p;
    const P* s = (const P*)st->h.s;
    const P* t = (const P*)st->h.t;
    const P* q = (const P*)st->h.q;
    C* x = (C*)st->h.x;
    C* pk = (C*)st->h.pk;
    double acc[1] = {0.0};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const P rv = ld_pack<false>(r + i), sv = ld_pack<false>(s + i), tv = ld_pack<false>(t + i);
        const P qv = ld_pack<false>(q + i);
        P pv0 = ld_pack<false>(p + i);
        P rn;
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            rn.v[e] = csub(sv.v[e], cmul(chi, tv.v[e]));
            pv0.v[e] = cadd(rn.v[e], cmul(alpha_new, csub(pv0.v[e], cmul(chi, qv.v[e]))));
            acc[0] += cnorm2(rn.v[e]);
        }
        for (int a0 = 0; a0 < na; a0 += UNR) {
            P xv[UNR], pv[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                if (a0 + u < na && !first) {
                    const int k = s_k[a0 + u];
                    xv[u] = ld_pack<true>((const P*)(x + k * n) + i);
                    pv[u] = ld_pack<true>((const P*)(pk + k * pks) + i);
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
                    st_pack<true>((P*)(x + k * n) + i, xo);
                    st_pack<true>((P*)(pk + k * pks) + i, po);
                }
            }
        }
        st_pack<false>(r + i, rn);
        st_pack<false>(p + i, pv0);
    }
    __shared__ double red[32];
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) {
        st->partial[blockIdx.x] = acc[0];
        if (blockIdx.x == 0) st->partial_count = gridDim.x;
    }
}

// end of iteration: |r'|^2 -> shuffle zeta/rho/delta/alpha/beta, per-shift stop test, loop control.
__global__ void __launch_bounds__(kThreads) k_bi_scal3(SolveState* st, cudaGraphConditionalHandle cond, int use_cond) {
    if (st->res.done) { if (use_cond && threadIdx.x == 0) cudaGraphSetConditional(cond, 0); return; }
    __shared__ double red[32];
    double s[1];
    reduce_partials<1>(st, s, red);
    const double rr = s[0];
    const int na = st->res.nactive;
    const int it = st->res.n_iter + 1;
    const double rnorm = sqrt(rr), bnorm = st->bnorm, tol = st->h.tol;
    const bool force = st->h.force_all != 0, base_rule = st->h.stop_rule == 1, psn = st->h.per_shift_norm != 0;
    for (int a = threadIdx.x; a < na; a += blockDim.x) {
        const int k = st->active[a];
        const zd zn = st->zeta_new[k], rn = st->rho_new[k];
        st->zeta_prev[k] = st->zeta[k];
        st->zeta[k] = zn;
        st->rho[k] = rn;
        const double zr = zabs(zmul(zn, rn));
        const double nk = psn ? st->rhs_norm[k] : bnorm;
        st->res.relres[k] = zr * rnorm / nk;
        if (!force && (base_rule ? rnorm : zr * rnorm) <= tol * nk) st->res.conv_iter[k] = it;
    }
    // msolve_set_history: row it-1 = beta, chi, alpha' (complex), |r'|^2, 0, then zeta_new[S], beta_k[S], chi_k[S] (complex)
    if (st->h.hist && it <= st->h.hist_cap) {
        __syncthreads();
        const int S = st->h.S;
        double* h = st->h.hist + (size_t)(it - 1) * (size_t)(8 + 6 * S);
        if (threadIdx.x == 0) {
            h[0] = st->beta.re; h[1] = st->beta.im; h[2] = st->chi.re; h[3] = st->chi.im;
            h[4] = st->alpha_new.re; h[5] = st->alpha_new.im; h[6] = rr; h[7] = 0.0;
        }
        for (int k = threadIdx.x; k < S; k += blockDim.x) {
            h[8 + 2 * k] = st->zeta_new[k].re; h[8 + 2 * k + 1] = st->zeta_new[k].im;
            h[8 + 2 * S + 2 * k] = st->beta_k[k].re; h[8 + 2 * S + 2 * k + 1] = st->beta_k[k].im;
            h[8 + 4 * S + 2 * k] = st->chi_k[k].re; h[8 + 4 * S + 2 * k + 1] = st->chi_k[k].im;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        st->R1 = rr;
        st->delta = st->delta_new;
        st->alpha = st->alpha_new;
        st->beta_prev = st->beta;
        st->res.n_iter = it;
        finish_iteration(st, !isfinite(rr));
        if (use_cond) cudaGraphSetConditional(cond, st->res.done ? 0u : 1u);
    }
}

}  // namespace msolve
