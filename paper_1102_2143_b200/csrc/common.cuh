// common.cuh -- shared device helpers for the msolve kernels (sm_100a).
// Complex arithmetic on interleaved (re,im) pairs, streaming load/store wrappers, deterministic
// block reductions and the device-resident solver state (the zeta /
// alpha / beta recurrences never leave the GPU).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/msolve.h"

namespace msolve {

constexpr int kMaxShifts = MSOLVE_MAX_SHIFTS;
constexpr int kMaxPartials = 4096;  // upper bound on any reducing kernel's grid size
constexpr int kAccMax = 5;          // doubles reduced per CTA (BiCGStab-M SpMV#2 needs 5)
constexpr int kThreads = 256;

// which vectors an SpMV launch works on and which reductions it fuses (spmv.cuh)
enum { ROLE_CG = 0, ROLE_B1 = 1, ROLE_B2 = 2, ROLE_GEN = 3 };

// ----------------------------------------------------------------------------- element types
// The kernels are templated on the ELEMENT type E of matrices and vectors: float2 / double2 are
// interleaved complex (MSOLVE_C64 / MSOLVE_C128, the BASELINE configs), float / double are real
// (MSOLVE_F32 / MSOLVE_F64, the paper's own runs, Table 1).  RealOf<E>::type is
// the precision T the vector arithmetic is done in; recurrence scalars are always fp64.
template <typename E> struct RealOf;
template <> struct RealOf<float>   { typedef float type; };
template <> struct RealOf<double>  { typedef double type; };
template <> struct RealOf<float2>  { typedef float type; };
template <> struct RealOf<double2> { typedef double type; };

template <typename C> __device__ __forceinline__ C cmake(double re, double im);
template <> __device__ __forceinline__ float2 cmake<float2>(double re, double im) { return make_float2((float)re, (float)im); }
template <> __device__ __forceinline__ double2 cmake<double2>(double re, double im) { return make_double2(re, im); }
// real data: every dot product is real, so the imaginary part of every scalar is exactly zero
template <> __device__ __forceinline__ float cmake<float>(double re, double) { return (float)re; }
template <> __device__ __forceinline__ double cmake<double>(double re, double) { return re; }

template <typename C> __device__ __forceinline__ C cadd(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) { C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r; }
// acc + a*b
template <typename C> __device__ __forceinline__ C cfma(C a, C b, C acc) {
    acc.x += a.x * b.x; acc.x -= a.y * b.y;
    acc.y += a.x * b.y; acc.y += a.y * b.x;
    return acc;
}
// a + s*b with real s
template <typename C, typename S> __device__ __forceinline__ C caxpy_r(C a, S s, C b) { C r; r.x = a.x + s * b.x; r.y = a.y + s * b.y; return r; }
// s*a + t*b with real s, t
template <typename C, typename S> __device__ __forceinline__ C clin_r(S s, C a, S t, C b) { C r; r.x = s * a.x + t * b.x; r.y = s * a.y + t * b.y; return r; }
// fp64 pieces of the fused reductions: |v|^2, Re / Im of conj(u) v
template <typename C> __device__ __forceinline__ double cnorm2(C v) { return (double)v.x * v.x + (double)v.y * v.y; }
template <typename C> __device__ __forceinline__ double cdot_re(C u, C v) { return (double)u.x * (double)v.x + (double)u.y * (double)v.y; }
template <typename C> __device__ __forceinline__ double cdot_im(C u, C v) { return (double)u.x * (double)v.y - (double)u.y * (double)v.x; }
template <typename C> __device__ __forceinline__ C cshfl_xor_add(C v, int o) {
    v.x += __shfl_xor_sync(0xffffffffu, v.x, o); v.y += __shfl_xor_sync(0xffffffffu, v.y, o); return v;
}

// real overloads (non-templates win overload resolution)
#define MSOLVE_REAL_OPS(R)                                                                          \
    __device__ __forceinline__ R cadd(R a, R b) { return a + b; }                                   \
    __device__ __forceinline__ R csub(R a, R b) { return a - b; }                                   \
    __device__ __forceinline__ R cmul(R a, R b) { return a * b; }                                   \
    __device__ __forceinline__ R cfma(R a, R b, R acc) { acc += a * b; return acc; }                \
    __device__ __forceinline__ R caxpy_r(R a, R s, R b) { return a + s * b; }                       \
    __device__ __forceinline__ R clin_r(R s, R a, R t, R b) { return s * a + t * b; }               \
    __device__ __forceinline__ double cnorm2(R v) { return (double)v * v; }                         \
    __device__ __forceinline__ double cdot_re(R u, R v) { return (double)u * (double)v; }           \
    __device__ __forceinline__ double cdot_im(R, R) { return 0.0; }                                 \
    __device__ __forceinline__ R cshfl_xor_add(R v, int o) { return v + __shfl_xor_sync(0xffffffffu, v, o); }
MSOLVE_REAL_OPS(float)
MSOLVE_REAL_OPS(double)
#undef MSOLVE_REAL_OPS

// ----------------------------------------------------------------------------- memory access
// Streaming (touched once per iteration, far larger than L2): evict-first loads / stores.
template <typename V> __device__ __forceinline__ V ld_stream(const V* p) { return __ldcs(p); }
template <typename V> __device__ __forceinline__ void st_stream(V* p, V v) { __stcs(p, v); }
// Read-only data reused by neighbouring rows / the next kernel: default caching, nc path.
template <typename V> __device__ __forceinline__ V ld_ro(const V* p) { return __ldg(p); }

// L2 cache policies for loads / bulk copies with a cache hint
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p; asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ uint64_t policy_evict_normal() {
    uint64_t p; asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p; asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p;
}
// Matrix stream: evict-first (read once per SpMV), or evict-last for `keep_pct` percent of the lines (chosen by the
// hardware from the address) and evict-first for the rest -- for a matrix of which only a part fits in L2 next to
// the vectors (MSOLVE_CFG_MATRIX_L2_KEEP_PERCENT).
__device__ __forceinline__ uint64_t policy_matrix(int keep_pct) {
    if (keep_pct <= 0) return policy_evict_first();
    if (keep_pct >= 100) return policy_evict_last();
    uint64_t p;
    const float f = 0.01f * (float)keep_pct;
    asm volatile("createpolicy.fractional.L2::evict_last.L2::evict_first.b64 %0, %1;" : "=l"(p) : "f"(f));
    return p;
}

// Gathered x of the CSR kernels, loaded with an L2 cache hint: evict_last pins x against the matrix
// stream when it fits in L2 comfortably (measured on config 5, B200: complex64, 34 MB of x: 0.98 ->
// 0.91 ms; complex128, 67 MB: 1.14 -> 1.34 ms, so there it is a plain ld.global.nc -- a hinted
// load with an evict_normal policy is slower than the plain one: 1.14 -> 1.38 ms).
template <bool PIN> __device__ __forceinline__ double2 ld_xg(const double2* p, uint64_t policy) {
    if (!PIN) return __ldg(p);
    double2 r; asm("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(r.x), "=d"(r.y) : "l"(p), "l"(policy)); return r;
}
template <bool PIN> __device__ __forceinline__ float2 ld_xg(const float2* p, uint64_t policy) {
    if (!PIN) return __ldg(p);
    float2 r; asm("ld.global.nc.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(r.x), "=f"(r.y) : "l"(p), "l"(policy)); return r;
}
template <bool PIN> __device__ __forceinline__ double ld_xg(const double* p, uint64_t policy) {
    if (!PIN) return __ldg(p);
    double r; asm("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(r) : "l"(p), "l"(policy)); return r;
}
template <bool PIN> __device__ __forceinline__ float ld_xg(const float* p, uint64_t policy) {
    if (!PIN) return __ldg(p);
    float r; asm("ld.global.nc.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(r) : "l"(p), "l"(policy)); return r;
}

// Matrix stream of the vector-CSR kernel (read once).  HINT: no L1 allocation + evict-first L2
// policy; used for elements of <= 8 bytes, where it is faster on B200 (config 5 complex64: 0.91 ->
// 0.73 ms); 16-byte elements are faster through a plain evict-first load (1.14 vs 1.34 ms).
#define MSOLVE_LD_MAT(TY, PTX, CONSTRAINT)                                                              \
    template <bool HINT> __device__ __forceinline__ TY ld_mat(const TY* p, uint64_t pol) {             \
        if (!HINT) return __ldcs(p);                                                                    \
        TY r; asm("ld.global.nc.L1::no_allocate.L2::cache_hint." PTX " %0, [%1], %2;" : CONSTRAINT(r) : "l"(p), "l"(pol)); return r; \
    }
MSOLVE_LD_MAT(int, "s32", "=r")
MSOLVE_LD_MAT(float, "f32", "=f")
MSOLVE_LD_MAT(double, "f64", "=d")
#undef MSOLVE_LD_MAT
template <bool HINT> __device__ __forceinline__ float2 ld_mat(const float2* p, uint64_t pol) {
    if (!HINT) return __ldcs(p);
    float2 r; asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(r.x), "=f"(r.y) : "l"(p), "l"(pol)); return r;
}
template <bool HINT> __device__ __forceinline__ double2 ld_mat(const double2* p, uint64_t) { return __ldcs(p); }

// ----------------------------------------------------------------------------- reductions
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Fixed-order CTA reduction of NACC doubles per thread; result valid in thread 0.
template <int NACC>
__device__ __forceinline__ void block_sum(double (&acc)[NACC], double* smem /* NACC * 32 */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = warp_sum(acc[a]);
    if (lane == 0) {
#pragma unroll
        for (int a = 0; a < NACC; ++a) smem[a * 32 + warp] = acc[a];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int a = 0; a < NACC; ++a) {
            double v = lane < nwarp ? smem[a * 32 + lane] : 0.0;
            acc[a] = warp_sum(v);
        }
    }
}

// ----------------------------------------------------------------------------- solver state
struct zd { double re, im; };  // complex double scalar on the device

__device__ __forceinline__ zd zmul(zd a, zd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ zd zadd(zd a, zd b) { return {a.re + b.re, a.im + b.im}; }
__device__ __forceinline__ zd zsub(zd a, zd b) { return {a.re - b.re, a.im - b.im}; }
__device__ __forceinline__ zd zneg(zd a) { return {-a.re, -a.im}; }
__device__ __forceinline__ zd zscale(zd a, double s) { return {a.re * s, a.im * s}; }
__device__ __forceinline__ zd zdiv(zd a, zd b) {  // Smith's algorithm
    if (fabs(b.re) >= fabs(b.im)) {
        const double r = b.im / b.re, d = b.re + b.im * r;
        return {(a.re + a.im * r) / d, (a.im - a.re * r) / d};
    }
    const double r = b.re / b.im, d = b.re * r + b.im;
    return {(a.re * r + a.im) / d, (a.im * r - a.re) / d};
}
__device__ __forceinline__ double zabs(zd a) { return hypot(a.re, a.im); }
__device__ __forceinline__ bool zfinite(zd a) { return isfinite(a.re) && isfinite(a.im); }
__device__ __forceinline__ bool zzero(zd a) { return a.re == 0.0 && a.im == 0.0; }

// Everything the iteration kernels need, resident in device memory for the whole solve.
// Pointers are read from here (not baked into kernel arguments) so one captured CUDA graph per
// handle serves every call.  Layout: [header: written by the host before a solve]
// [result: read back by the host after it] [device-only scratch].
struct SolveHeader {
    // vectors (complex<T>, T from the handle's dtype)
    const void* b;   // rhs; also the BiCGStab-M shadow vector r0
    void* x;         // [S][n] shift-major, caller's output
    void* r;         // base residual
    void* p;         // base search direction
    void* q;         // A p
    void* s;         // BiCGStab-M: s = r + beta q
    void* t;         // BiCGStab-M: t = A s
    void* pk;        // [S][pk_stride] per-shift search directions
    // generic SpMV roles (msolve_spmv)
    const void* sp_x; void* sp_y; const void* sp_u;
    long long n;
    long long pk_stride;
    long long x_stride;  // elements between x_k and x_{k+1} (n for a single handle; the global n for a slab, slab.cu)
    double tol;
    int S;
    int max_iter;
    int force_all;   // profiling: never converge, never stop before max_iter
    int stop_rule;   // 0 = per shift (R15), 1 = literal |r| > eps on the unshifted system (Alg. 1 l.15)
    double* hist;    // msolve_set_history: per-iteration scalars, hist_cap rows (NULL = off)
    int hist_cap;
    unsigned long long* phase_ns;   // msolve_set_phase_clock (one-kernel path), NULL = off
    int per_shift_norm;  // eq. (6): the stop test of shift k is relative to rhs_norm[k] = ||b_k|| instead of ||b||
    // deferred multishift update (CG-M, graph path; kernels.cuh "deferred update"): ring of defer + 1 residual vectors
    // (r itself lives in it), defer = chunk length M (0 = the classic update of every x_k, p_k in every iteration)
    void* ring;
    long long ring_stride;   // BYTES between two slots of the ring
    int defer;
    double sigma[kMaxShifts];
};

struct SolveResult {
    int n_iter;
    int done;
    int status;
    int nactive;
    int zero_rhs;
    int pad1;
    int conv_iter[kMaxShifts];
    double relres[kMaxShifts];
};

// The recurrence scalars of the iteration (Alg. 1 l.2-8, 17, 20-26, 30-31).  One instance lives in the
// device-resident SolveState (iteration as a graph of kernels); the whole-solve cooperative kernel
// (fused_small.cuh) keeps a private copy per CTA in shared memory.
struct Recur {
    // base scalars (CG-M uses .re only)
    zd alpha, beta, beta_prev, delta, chi, alpha_new, delta_new;
    double R0, R1, bnorm;
    // per shift
    zd zeta_prev[kMaxShifts], zeta[kMaxShifts], zeta_new[kMaxShifts];
    zd rho[kMaxShifts], rho_new[kMaxShifts];
    zd beta_k[kMaxShifts], alpha_k[kMaxShifts], chi_k[kMaxShifts];
    int active[kMaxShifts];      // compact list of active shift indices, length res.nactive
    // per-ACTIVE-shift coefficients consumed by the fused update kernels (index = position in
    // `active`): CG-M uses 3 reals (zeta, alpha_k, beta_k); BiCGStab-M 7 complex.
    double coef[kMaxShifts * 14];
};

// Deferred multishift update: bookkeeping of one chunk of at most kDeferMax iterations (kernels.cuh).  The shifts
// that were active when the chunk began are `list`; for list position a and chunk-relative iteration j
//   p_k(now)  = Ap[a] P_k + sum_j Cp[a][j] r_j,      x_k(now) = X_k + Ax[a] P_k + sum_j Cx[a][j] r_j
// with P_k, X_k the vectors in memory (written by the previous flush) and r_j the residuals kept in the ring.
constexpr int kDeferMax = 32;
struct Defer {
    int fill;            // residuals of the chunk whose coefficients are complete (= iterations done in the chunk)
    int s0;              // ring slot of the chunk's first residual
    int first;           // 1 until the first flush: P_k, X_k are not in memory yet (p_k(-1) = 0, x_k(0) = 0)
    int need_begin;      // the next scal1 starts a new chunk
    int nlist;
    unsigned int ticket; // last-CTA detection of the flush kernel
    void* r_next;        // where the r update of this iteration writes r_{n+1}
    int list[kMaxShifts];    // shift index of list position a
    int pos[kMaxShifts];     // list position of shift k
    double Ap[kMaxShifts], Ax[kMaxShifts];
    double Cp[kMaxShifts * kDeferMax], Cx[kMaxShifts * kDeferMax];
};

// one CTA's contribution to a grid-wide sum of the one-kernel path (fused_small.cu): values + generation tag
constexpr int kFusedMaxCtas = 160;
struct alignas(128) FusedSlot { unsigned long long w[2 * kAccMax]; unsigned long long tag; };

struct SolveState {
    SolveHeader h;
    SolveResult res;
    Recur rc;
    double rhs_norm[kMaxShifts]; // eq. (6) only: ||b_k|| (multirhs.cu)
    // per-CTA partial sums of the fused reductions, [kAccMax][kMaxPartials]
    double partial[kAccMax * kMaxPartials];
    int partial_count;           // how many CTAs wrote partials in the last reducing kernel
    // fused_small.cu: slots of the combined grid barrier + sum, double-buffered by the parity of the generation
    // counter, which runs on from solve to solve (fused_gen)
    FusedSlot fslot[2][kFusedMaxCtas];
    unsigned long long fused_gen;
    Defer df;
};

// Fixed-order reduction of `count` per-CTA partials (NACC rows of kMaxPartials) by ONE CTA: every thread of the
// calling CTA gets the sums (deterministic for a fixed grid).
template <int NACC>
__device__ __forceinline__ void reduce_partials_from(const double* partial, int count, double (&out)[NACC], double* smem) {
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    for (int i = threadIdx.x; i < count; i += blockDim.x) {
#pragma unroll
        for (int a = 0; a < NACC; ++a) acc[a] += partial[a * kMaxPartials + i];
    }
    block_sum<NACC>(acc, smem);
    __shared__ double bc[kAccMax];
    __syncthreads();                     // bc may still be read from a previous call
    if (threadIdx.x == 0) {
#pragma unroll
        for (int a = 0; a < NACC; ++a) bc[a] = acc[a];
    }
    __syncthreads();
#pragma unroll
    for (int a = 0; a < NACC; ++a) out[a] = bc[a];
}
template <int NACC>
__device__ __forceinline__ void reduce_partials(const SolveState* st, double (&out)[NACC], double* smem) {
    reduce_partials_from<NACC>(st->partial, st->partial_count, out, smem);
}

// Matrix description passed by value to the SpMV kernels.
struct MatDev {
    const int32_t* rowptr;   // CSR: n+1 ; BSR3: nbrows+1
    const int32_t* colidx;   // CSR: nnz ; BSR3: nblocks (block column)
    const void* val;         // CSR: nnz complex ; BSR3: nblocks*9 complex
    long long n;             // scalar rows
    long long nbrows;        // BSR3 block rows (0 for CSR)
    long long nnz;           // CSR nnz / BSR3 blocks
    const int32_t* aux;      // merge-path partition table / BSR tile table
    void* carry;             // merge-path: per-tile head / tail partial sums, 2 * aux_count complex
    int aux_count;
    int x_pin;               // CSR kernels: gather x with L2 evict_last (x fits in L2 next to the stream)
    int mat_keep;            // percent of the matrix stream loaded with L2 evict_last (0: all evict-first), policy_matrix()
    // matrix-free SU(3) lattice operator (msolve_create_lattice_su3): val = links[ndim][vol][3][3]
    int lat_ndim;            // 0 for CSR / BSR3
    int lat_ext[4];          // extents, dimension 0 fastest (unused dimensions = 1)
    int lat_rows_per_tile;   // x0-rows per tile of the TMA kernel
    long long lat_vol;       // number of sites
    double lat_diag, lat_cf, lat_cb;
};

}  // namespace msolve
