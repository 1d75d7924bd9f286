// resident.cu -- CG-M and BiCGStab-M with the whole problem resident in SHARED MEMORY (BASELINE configs 1-2 and the like).
//
// A B200 has 148 SMs x 227 KB = 33 MB of shared memory.  When the matrix and all 3 + 2S vectors of the solve fit
// there, one persistent cooperative kernel gives every CTA a contiguous range of rows and keeps, for the whole
// solve, that range of the matrix and of r, p, Ap and every x_k, p_k in its shared memory.  Per iteration the only
// global-memory traffic is the exchange the method itself needs: the search direction p (written by its owner,
// gathered by the rows that reference it: the "halo") and the two dot products (fused_allreduce: one round trip to
// L2 each, no atomics).  Everything else -- the matrix stream and the 4S + 3 vector passes of the fused multishift
// update (Alg. 1 l.21, 24, 28, 29) -- runs out of shared memory.  x_k is written to the caller's
// array once, at the end.
//
// Same steps, same per-element arithmetic and the same scalar functions (kernels.cuh) as the other two paths; the
// dot products are grouped by row owner, so results agree with them to rounding and are bit-reproducible.
// One thread per scalar row of the CTA's range (CSR: the row's non-zeros in stored order; BSR3: row r of each 3x3
// block of the block row).
#include "handle.h"
#include "tuning.h"
#include "kernels.cuh"
#include "fused_sync.cuh"

namespace msolve {

constexpr int kResThreads = 256;

// layout of a CTA's dynamic shared memory (byte offsets, the same in every CTA: sized for the largest range)
struct ResLayout {
    int max_rows;        // scalar rows per CTA (upper bound)
    int max_units;       // index rows per CTA: scalar rows (CSR) or block rows (BSR3)
    int max_entries;     // non-zeros (CSR) or blocks (BSR3) per CTA
    int off_rowptr, off_col, off_val, off_r, off_p, off_q, off_s, off_t, off_b, off_xk, off_pk;   // s, t, b: BiCGStab-M only
    int S;
    int total;
};

// (A x)_i for local scalar row i: matrix out of shared memory, x gathered from global memory
template <typename C, int DOF>
__device__ __forceinline__ C res_row_product(int i, const int* s_rowptr, const int* s_col, const C* s_val, const C* xg) {
    C sum = cmake<C>(0.0, 0.0);
    if (DOF == 3) {
        const int lbr = i / 3, rr = i - 3 * lbr;
        for (int j = s_rowptr[lbr]; j < s_rowptr[lbr + 1]; ++j) {
            const C* blk = s_val + j * 9 + rr * 3;
            const C* xv = xg + 3ll * s_col[j];
            sum = cfma(blk[0], xv[0], sum);
            sum = cfma(blk[1], xv[1], sum);
            sum = cfma(blk[2], xv[2], sum);
        }
    } else {
#pragma unroll 4
        for (int j = s_rowptr[i]; j < s_rowptr[i + 1]; ++j) sum = cfma(s_val[j], xg[s_col[j]], sum);
    }
    return sum;
}

// what both kernels start with: private state, the CTA's range, its slice of the matrix into shared memory
#define MSOLVE_RESIDENT_PROLOGUE                                                                        \
    typedef E C;                                                                                        \
    typedef typename RealOf<E>::type T;                                                                 \
    extern __shared__ __align__(16) unsigned char dyn[];                                                \
    Recur& rc = *(Recur*)dyn;                                                                           \
    SolveResult& res = *(SolveResult*)(dyn + kFusedOffRes);                                             \
    const SolveHeader& h = *(const SolveHeader*)(dyn + kFusedOffHdr);                                   \
    double* rhs_norm = (double*)(dyn + kFusedOffNorm);                                                  \
    unsigned char* base = dyn + kFusedFixedBytes;                                                       \
    __shared__ double red[kAccMax * 32];                                                                \
    fused_stage_header(hp, st, dyn + kFusedOffHdr, rhs_norm);                                               \
    const int cta = blockIdx.x, ncta = gridDim.x, tid = threadIdx.x;                                    \
    const long long units = DOF == 3 ? A.nbrows : A.n;                                                  \
    const long long u0 = units * cta / ncta, u1 = units * (cta + 1) / ncta;                             \
    const int nu = (int)(u1 - u0), nloc = nu * DOF;                                                     \
    const long long row0 = u0 * DOF;                                                                    \
    int* s_rowptr = (int*)(base + L.off_rowptr);                                                        \
    int* s_col = (int*)(base + L.off_col);                                                              \
    C* s_val = (C*)(base + L.off_val);                                                                  \
    C* s_r = (C*)(base + L.off_r);                                                                      \
    C* s_p = (C*)(base + L.off_p);                                                                      \
    C* s_q = (C*)(base + L.off_q);                                                                      \
    C* s_xk = (C*)(base + L.off_xk);     /* [S][max_rows] */                                            \
    C* s_pk = (C*)(base + L.off_pk);                                                                    \
    const int ld = L.max_rows;                                                                          \
    const int S = h.S;                                                                                  \
    C* pg = (C*)h.p;                     /* lives in global memory: gathered across CTAs */              \
    {                                                                                                   \
        const int e0 = A.rowptr[u0];                                                                    \
        const int ne = A.rowptr[u1] - e0;                                                               \
        for (int i = tid; i <= nu; i += blockDim.x) s_rowptr[i] = A.rowptr[u0 + i] - e0;                \
        for (int j = tid; j < ne; j += blockDim.x) s_col[j] = A.colidx[e0 + j];                         \
        const C* gv = (const C*)A.val + (long long)e0 * (DOF == 3 ? 9 : 1);                             \
        const int nv = ne * (DOF == 3 ? 9 : 1);                                                         \
        for (int j = tid; j < nv; j += blockDim.x) s_val[j] = gv[j];                                    \
    }                                                                                                   \
    (void)sizeof(T); (void)cta

// the solutions leave shared memory once
#define MSOLVE_RESIDENT_EPILOGUE                                                                        \
    {                                                                                                   \
        C* x = (C*)h.x;                                                                                 \
        const long long xs = h.x_stride;                                                                \
        const bool none = res.n_iter == 0;   /* stopped before the first update: x_k = 0 */             \
        for (int i = tid; i < nloc; i += blockDim.x)                                                    \
            for (int k = 0; k < S; ++k) x[k * xs + row0 + i] = none ? cmake<C>(0.0, 0.0) : s_xk[k * ld + i]; \
    }                                                                                                   \
    fused_publish(st, res, gen)

// p_n = r_n + alpha_n p_{n-1}, with explicit fused multiply-adds: the owner of a row and every CTA that gathers the
// row evaluate this same expression on the same operands and must get the same bits
__device__ __forceinline__ double2 res_pnext(double2 r, double a, double2 p) { return make_double2(fma(a, p.x, r.x), fma(a, p.y, r.y)); }
__device__ __forceinline__ float2 res_pnext(float2 r, float a, float2 p) { return make_float2(fmaf(a, p.x, r.x), fmaf(a, p.y, r.y)); }
__device__ __forceinline__ double res_pnext(double r, double a, double p) { return fma(a, p, r); }
__device__ __forceinline__ float res_pnext(float r, float a, float p) { return fmaf(a, p, r); }

// (A p_n)_i with p_n = r_n + alpha_n p_{n-1} formed on the fly from the two vectors that ARE visible in global memory
template <typename C, typename T, int DOF>
__device__ __forceinline__ C res_row_product_pnext(int i, const int* s_rowptr, const int* s_col, const C* s_val, const C* rg,
                                                   const C* pold, T alpha) {
    C sum = cmake<C>(0.0, 0.0);
    if (DOF == 3) {
        const int lbr = i / 3, rr = i - 3 * lbr;
        for (int j = s_rowptr[lbr]; j < s_rowptr[lbr + 1]; ++j) {
            const C* blk = s_val + j * 9 + rr * 3;
            const long long c = 3ll * s_col[j];
            sum = cfma(blk[0], res_pnext(rg[c], alpha, pold[c]), sum);
            sum = cfma(blk[1], res_pnext(rg[c + 1], alpha, pold[c + 1]), sum);
            sum = cfma(blk[2], res_pnext(rg[c + 2], alpha, pold[c + 2]), sum);
        }
    } else {
#pragma unroll 4
        for (int j = s_rowptr[i]; j < s_rowptr[i + 1]; ++j) {
            const int c = s_col[j];
            sum = cfma(s_val[j], res_pnext(rg[c], alpha, pold[c]), sum);
        }
    }
    return sum;
}

// CG-M.  Two grid-wide exchanges per iteration, the two sums the method needs (<p,Ap> and |r|^2): the search
// direction is never waited for.  Owners mirror r (written during the update, i.e. before the |r|^2 sum) and p
// (two buffers in turn, written right after alpha is known) in global memory; a CTA that gathers column j in
// iteration n forms p_n[j] = r_n[j] + alpha_n p_{n-1}[j] itself from r_n and p_{n-1}, both of which became visible
// with sums it has already passed.  The buffer p_n is written into was last read two sums ago.
template <typename E, int DOF>
__global__ void __launch_bounds__(kResThreads, 1) k_cgm_resident(MatDev A, SolveState* st, ResLayout L, const __grid_constant__ SolveHeader hp) {
    MSOLVE_RESIDENT_PROLOGUE;
    C* rg = (C*)h.r;                                          // mirror of r
    C* pbuf[2] = {pg, (C*)h.q};                               // mirrors of p_n (n even / odd); q itself stays in shared memory
    // r <- b, p <- b, x_k <- 0, p_k <- b  (l.9-12)
    double acc[1] = {0.0}, s[1];
    for (int i = tid; i < nloc; i += blockDim.x) {
        const C bv = ((const C*)h.b)[row0 + i];
        s_r[i] = bv; s_p[i] = bv;
        pbuf[0][row0 + i] = bv;
        rg[row0 + i] = bv;
        for (int k = 0; k < S; ++k) { s_xk[k * ld + i] = cmake<C>(0.0, 0.0); s_pk[k * ld + i] = bv; }
        acc[0] += cnorm2(bv);
    }
    unsigned long long gen = st->fused_gen;
    fused_allreduce<1>(st, gen, acc, s, red);                                        // <b,b> (l.13); p_0, r_0 visible to all
    init_state_fn(h, res, rc, s[0]);
    while (!res.done) {
        const int n = res.n_iter;
        const T alpha = (T)rc.alpha.re;
        acc[0] = 0.0;
        if (n > 0) {
            C* pnew = pbuf[n & 1];
            const C* pold = pbuf[(n - 1) & 1];
            for (int i = tid; i < nloc; i += blockDim.x) {                           // l.27, own rows; nobody waits for this store
                const C pv = res_pnext(s_r[i], alpha, s_p[i]);
                s_p[i] = pv;
                pnew[row0 + i] = pv;
            }
            __syncthreads();
            for (int i = tid; i < nloc; i += blockDim.x) {                           // l.18-19
                const C sum = res_row_product_pnext<C, T, DOF>(i, s_rowptr, s_col, s_val, rg, pold, alpha);
                s_q[i] = sum;
                acc[0] += cdot_re(s_p[i], sum);
            }
        } else {
            for (int i = tid; i < nloc; i += blockDim.x) {
                const C sum = res_row_product<C, DOF>(i, s_rowptr, s_col, s_val, pbuf[0]);
                s_q[i] = sum;
                acc[0] += cdot_re(s_p[i], sum);
            }
        }
        fused_allreduce<1>(st, gen, acc, s, red);
        cgm_scal1_fn(h, res, rc, s[0]);                                               // l.20, 22, 23
        if (res.done) break;
        {                                                                             // l.21, 24, 28, 29 out of shared memory
            const int na = res.nactive;
            const T beta = (T)rc.beta.re;
            acc[0] = 0.0;
            for (int i = tid; i < nloc; i += blockDim.x) {
                C rv = s_r[i];
                for (int a = 0; a < na; ++a) {
                    const int k = rc.active[a];
                    const T zk = (T)rc.coef[3 * a + 0], ak = (T)rc.coef[3 * a + 1], bk = (T)rc.coef[3 * a + 2];
                    const C pe = clin_r(zk, rv, ak, s_pk[k * ld + i]);                // l.29 (lagged); n = 0: zk = 1, ak = 0
                    s_xk[k * ld + i] = caxpy_r(s_xk[k * ld + i], -bk, pe);            // l.28
                    s_pk[k * ld + i] = pe;
                }
                rv = caxpy_r(rv, beta, s_q[i]);                                       // l.21
                s_r[i] = rv;
                rg[row0 + i] = rv;                                                    // visible with the |r|^2 sum
                acc[0] += cnorm2(rv);                                                 // l.24
            }
        }
        fused_allreduce<1>(st, gen, acc, s, red);
        cgm_scal2_fn(h, res, rc, rhs_norm, s[0], cta == 0 ? h.hist : nullptr);        // l.25, 26, 30, 31, 15
    }
    MSOLVE_RESIDENT_EPILOGUE;
}

// BiCGStab-M, same residency: r, p, q, s, t, b and every x_k, p_k in shared memory; p and s are the two vectors the
// SpMVs gather, so they are mirrored in global memory.  Steps and per-element arithmetic of k_bi_fused / bi_update_fn.
template <typename E, int DOF>
__global__ void __launch_bounds__(kResThreads, 1) k_bi_resident(MatDev A, SolveState* st, ResLayout L, const __grid_constant__ SolveHeader hp) {
    MSOLVE_RESIDENT_PROLOGUE;
    C* s_s = (C*)(base + L.off_s);
    C* s_t = (C*)(base + L.off_t);
    C* s_b = (C*)(base + L.off_b);
    C* sg = (C*)h.s;
    __shared__ C s_c[kMaxShifts * 7];
    double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, s[5];
    for (int i = tid; i < nloc; i += blockDim.x) {
        const C bv = ((const C*)h.b)[row0 + i];
        s_r[i] = bv; s_p[i] = bv; s_b[i] = bv;
        pg[row0 + i] = bv;
        for (int k = 0; k < S; ++k) { s_xk[k * ld + i] = cmake<C>(0.0, 0.0); s_pk[k * ld + i] = bv; }
        acc[0] += cnorm2(bv);
    }
    unsigned long long gen = st->fused_gen;
    fused_allreduce<1>(st, gen, acc, s, red);
    init_state_fn(h, res, rc, s[0]);
    while (!res.done) {
        acc[0] = acc[1] = 0.0;
        for (int i = tid; i < nloc; i += blockDim.x) {                               // q = A p, <r0,q>
            const C sum = res_row_product<C, DOF>(i, s_rowptr, s_col, s_val, pg);
            s_q[i] = sum;
            acc[0] += cdot_re(s_b[i], sum);
            acc[1] += cdot_im(s_b[i], sum);
        }
        fused_allreduce<2>(st, gen, acc, s, red);
        bi_scal1_fn(h, res, rc, zd{s[0], s[1]});
        if (res.done) break;
        {
            const C beta = cmake<C>(rc.beta.re, rc.beta.im);
            for (int i = tid; i < nloc; i += blockDim.x) {                           // s = r + beta q
                const C sv = cfma(beta, s_q[i], s_r[i]);
                s_s[i] = sv;
                sg[row0 + i] = sv;
            }
        }
        fused_allreduce<0>(st, gen, nullptr, nullptr, red);                          // s complete before it is gathered
#pragma unroll
        for (int a = 0; a < 5; ++a) acc[a] = 0.0;
        for (int i = tid; i < nloc; i += blockDim.x) {                               // t = A s, <t,s>, <t,t>, <r0,t>
            const C sum = res_row_product<C, DOF>(i, s_rowptr, s_col, s_val, sg);
            s_t[i] = sum;
            const C xi = s_s[i], ui = s_b[i];
            acc[0] += cdot_re(sum, xi);
            acc[1] += cdot_im(sum, xi);
            acc[2] += cnorm2(sum);
            acc[3] += cdot_re(ui, sum);
            acc[4] += cdot_im(ui, sum);
        }
        fused_allreduce<5>(st, gen, acc, s, red);
        bi_scal2_fn(h, res, rc, s);
        if (res.done) break;
        {
            const int na = res.nactive;
            for (int j = tid; j < 7 * na; j += blockDim.x) s_c[j] = cmake<C>(rc.coef[2 * j], rc.coef[2 * j + 1]);
            const C chi = cmake<C>(rc.chi.re, rc.chi.im);
            const C alpha_new = cmake<C>(rc.alpha_new.re, rc.alpha_new.im);
            __syncthreads();
            acc[0] = 0.0;
            for (int i = tid; i < nloc; i += blockDim.x) {                           // r', p, x_k, p_k, |r'|^2
                const C rv = s_r[i], sv = s_s[i];
                const C rn = csub(sv, cmul(chi, s_t[i]));
                const C pn = cadd(rn, cmul(alpha_new, csub(s_p[i], cmul(chi, s_q[i]))));
                acc[0] += cnorm2(rn);
                for (int a = 0; a < na; ++a) {
                    const int k = rc.active[a];
                    const C* c = s_c + 7 * a;
                    const C pe = s_pk[k * ld + i];
                    s_xk[k * ld + i] = cadd(csub(s_xk[k * ld + i], cmul(c[0], pe)), cmul(c[1], sv));
                    const C ds = csub(cmul(c[5], sv), cmul(c[6], rv));
                    s_pk[k * ld + i] = cadd(cmul(c[2], rn), cmul(c[3], csub(pe, cmul(c[4], ds))));
                }
                s_r[i] = rn;
                s_p[i] = pn;
                pg[row0 + i] = pn;
            }
        }
        fused_allreduce<1>(st, gen, acc, s, red);                                    // also: p complete before SpMV#1
        bi_scal3_fn(h, res, rc, rhs_norm, s[0], cta == 0 ? h.hist : nullptr);
    }
    MSOLVE_RESIDENT_EPILOGUE;
}

// ------------------------------------------------------------------------------------------- host side
static int res_dof(const msolve_matrix* A) { return A->format == FMT_BSR3 ? 3 : 1; }

// Sizes the shared-memory layout for `ncta` CTAs; false when a CTA's range does not fit.
static bool resident_layout(const msolve_matrix* A, int S, int alg, int ncta, ResLayout* L) {
    const int dof = res_dof(A);
    const long long units = dof == 3 ? A->dev.nbrows : A->dev.n;
    if ((long long)A->h_rowptr.size() != units + 1) return false;
    long long max_units = 0, max_entries = 0;
    for (int c = 0; c < ncta; ++c) {
        const long long u0 = units * c / ncta, u1 = units * (c + 1) / ncta;
        max_units = std::max(max_units, u1 - u0);
        if (A->h_rowptr[u1] < A->h_rowptr[u0]) return false;             // not a CSR row pointer: leave it to the other paths
        max_entries = std::max<long long>(max_entries, A->h_rowptr[u1] - A->h_rowptr[u0]);
    }
    const size_t e = elem_bytes(A->dtype);
    auto up = [](size_t v) { return (v + 15) / 16 * 16; };
    size_t off = 0;
    L->max_units = (int)max_units; L->max_rows = (int)(max_units * dof); L->max_entries = (int)max_entries; L->S = S;
    L->off_rowptr = (int)off; off += up(sizeof(int) * (size_t)(max_units + 1));
    L->off_col = (int)off; off += up(sizeof(int) * (size_t)max_entries);
    L->off_val = (int)off; off += up(e * (size_t)max_entries * (dof == 3 ? 9 : 1));
    const size_t vec = up(e * (size_t)L->max_rows);
    L->off_r = (int)off; off += vec;
    L->off_p = (int)off; off += vec;
    L->off_q = (int)off; off += vec;
    L->off_s = L->off_t = L->off_b = 0;
    if (alg == MSOLVE_ALG_BICGSTABM) {
        L->off_s = (int)off; off += vec;
        L->off_t = (int)off; off += vec;
        L->off_b = (int)off; off += vec;
    }
    L->off_xk = (int)off; off += (size_t)S * e * (size_t)L->max_rows;
    off = up(off);
    L->off_pk = (int)off; off += (size_t)S * e * (size_t)L->max_rows;
    const size_t fixed = (size_t)kFusedFixedBytes;
    if (off + fixed > (size_t)200 * 1024) return false;
    L->total = (int)(off + fixed);
    return true;
}

bool resident_supported(const msolve_matrix* A, int S, int alg) {
    if (A->format != FMT_CSR && A->format != FMT_BSR3) return false;
    if (A->opt.update_kernel != 0 || A->opt.loop_mode != 0 || A->dev.n == 0) return false;
    int coop = 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, A->device) != cudaSuccess || !coop) return false;
    ResLayout L;
    return resident_layout(A, S, alg, std::min(A->num_sms, kFusedMaxCtas), &L);
}

template <typename E, int DOF>
static int launch_resident_t(const msolve_matrix* A, int alg, const ResLayout& L, int ncta, cudaStream_t s) {
    auto kernel = alg == MSOLVE_ALG_CGM ? k_cgm_resident<E, DOF> : k_bi_resident<E, DOF>;
    int rc = ensure_smem(A, (const void*)kernel, L.total);
    if (rc != MSOLVE_OK) return rc;
    MatDev dev = A->dev;
    SolveState* st = A->d_state;
    ResLayout lay = L;
    SolveHeader hdr = A->h_stage->h;
    void* args[4] = {&dev, &st, &lay, &hdr};
    MSOLVE_CU(cudaLaunchCooperativeKernel((const void*)kernel, dim3(ncta), dim3(kResThreads), args, (size_t)L.total, s));
    return MSOLVE_OK;
}

int launch_resident(const msolve_matrix* A, int S, int alg, cudaStream_t s) {
    const int ncta = std::min(A->num_sms, kFusedMaxCtas);
    ResLayout L;
    if (!resident_layout(A, S, alg, ncta, &L)) return fail(MSOLVE_EINVAL, "resident path: the problem does not fit in shared memory");
    const bool bsr = A->format == FMT_BSR3;
    switch (A->dtype) {
        case MSOLVE_C128: return bsr ? launch_resident_t<double2, 3>(A, alg, L, ncta, s) : launch_resident_t<double2, 1>(A, alg, L, ncta, s);
        case MSOLVE_C64:  return bsr ? launch_resident_t<float2, 3>(A, alg, L, ncta, s) : launch_resident_t<float2, 1>(A, alg, L, ncta, s);
        case MSOLVE_F64:  return launch_resident_t<double, 1>(A, alg, L, ncta, s);
        default:          return launch_resident_t<float, 1>(A, alg, L, ncta, s);
    }
}

}  // namespace msolve
