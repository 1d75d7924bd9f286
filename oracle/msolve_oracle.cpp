// msolve_oracle.cpp -- CPU ORACLE for the multishift Krylov solvers CG-M and BiCGStab-M.
//
// TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code
// with the CUDA path (paper_1102_2143_b200/csrc): no common headers, helpers or constants.
//
// What it is: a plain, slow, single-threaded, step-by-step restatement of
//   * eq. (1), PAPER.md:41          (A + sigma_k I) x_k = b            -- the result
//   * Algorithm 1, PAPER.md:73-142  CG-M, with the garbled lines read as SURVEY.md 8(c) C2
//                                   (R2-R7)
//   * BiCGStab-M, named at PAPER.md:31,154 and attributed to [4] PAPER.md:244; the paper never
//     prints it, so it is derived from the collinear-residual argument (eq. (4))
//     as SURVEY.md 8(c) C3 / DESIGN.md "BiCGStab-M derivation".
//   * plain CG and plain BiCGStab (textbook, van der Vorst [13] PAPER.md:253) used ONLY as the
//     sigma=0 / single-shift pins of the two multishift routines.
// No blocking, fusion or reordering: every loop below is one line of the algorithm.
//
// Precision (R14): vectors are complex<T> or, for the paper's own real-valued workload
// (Table 1), plain T; T = float or double; every
// dot product accumulates in double, every recurrence scalar (zeta, alpha, beta, rho, chi) is
// double / complex<double>; a scalar that multiplies a vector is rounded to T once, then the
// vector arithmetic is done in T.  SpMV accumulates a row in T in stored order.
//
// Pins (tests/test_oracle_pins.py, run with -m "not gpu"): dense LU of (A+sigma I) on tiny
// inputs, A = c*I closed form, diagonal-A finite termination, per-iteration collinearity
// invariant b-(A+sigma)x_k = zeta_k r (CG-M) / zeta_k rho_k r (BiCGStab-M), sigma=0 reduction to
// plain CG (bitwise) / plain BiCGStab, independent single-shift solves, FFT closed form on a
// pure-gauge SU(3) lattice, sine-transform closed form on the paper's 2-D Poisson matrix,
// monotone conv_iter in sigma, true residual <= tol.  Nothing here is "parity unpinned";
// the choice of stop/mask rule (R15) is a reading, pinned only as oracle == GPU.
//
// Build: g++ -O2 -ffp-contract=off -shared -fPIC (see oracle/__init__.py).
// The `#pragma omp` lines are inert in that build (no -fopenmp): the parity oracle is single-threaded and
// every sum has one fixed order.  oracle.build_omp() compiles the SAME source with -fopenmp into a second
// library used only by bench.py's cpu_baseline / --impl reference timing legs (all host cores; its dot
// products are summed per thread, so it is not the parity configuration).

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

typedef std::complex<double> zdouble;

enum { ST_OK = 0, ST_MAXITER = 1, ST_BREAKDOWN = 2, ST_EINVAL = -1 };

// Element type C of matrices and vectors: std::complex<T> (the BASELINE configs) or plain T (the
// paper's own real-valued runs, Table 1); T = float or double.
template <typename C> struct RealOf { typedef C type; };
template <typename T> struct RealOf<std::complex<T> > { typedef T type; };

template <typename C>
struct Csr {
    int64_t n;
    const int32_t* rowptr;
    const int32_t* colidx;
    const C* val;
};

// y = A x   (Alg. 1 l.18).  Row sum in T, stored order.
template <typename C>
void spmv(const Csr<C>& A, const C* x, C* y) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < A.n; ++i) {
        C acc(0);
        for (int32_t j = A.rowptr[i]; j < A.rowptr[i + 1]; ++j) acc += A.val[j] * x[A.colidx[j]];
        y[i] = acc;
    }
}

// <u,v> = sum_i conj(u_i) v_i, accumulated in double (r^dagger . r).
template <typename C>
zdouble dot(int64_t n, const C* u, const C* v) {
    double re = 0.0, im = 0.0;                      // the two components of one complex accumulator
#pragma omp parallel for schedule(static) reduction(+ : re, im)
    for (int64_t i = 0; i < n; ++i) {
        const zdouble t = std::conj(zdouble(u[i])) * zdouble(v[i]);
        re += t.real();
        im += t.imag();
    }
    return zdouble(re, im);
}

// A recurrence scalar rounded ONCE to the vectors' element type (R14).  Real data: every dot
// product is real, so every scalar has an exactly zero imaginary part and the real part is it.
template <typename C> struct Rnd;
template <typename T> struct Rnd<std::complex<T> > {
    static std::complex<T> of(const zdouble& z) { return std::complex<T>((T)z.real(), (T)z.imag()); }
};
template <> struct Rnd<float> { static float of(const zdouble& z) { return (float)z.real(); } };
template <> struct Rnd<double> { static double of(const zdouble& z) { return z.real(); } };
template <typename C> inline C rnd(const zdouble& z) { return Rnd<C>::of(z); }
template <typename C> inline C rnd(double v) { return Rnd<C>::of(zdouble(v, 0)); }

inline bool finite(double x) { return std::isfinite(x); }
inline bool finite(const zdouble& z) { return std::isfinite(z.real()) && std::isfinite(z.imag()); }

// ------------------------------------------------------------------------------------------
// CG-M.  Alg. 1 with the readings of DESIGN.md R2-R7:
//   beta = -R0/P (sign restored), zeta recurrence with beta_prev and alpha,
//   beta_k = beta zeta_new/zeta, alpha_k = alpha (zeta_new/zeta)^2, p_k uses zeta_new and new r.
// Stop / mask rule R15: shift k is frozen at the first n with |zeta_k| ||r|| <= tol ||b||.
// hist (optional, hist_cap rows of 3+3S doubles): per iteration beta, alpha_next, R1 and per
// shift zeta_new, beta_k, alpha_k.
// ------------------------------------------------------------------------------------------
template <typename C>
int cgm(const Csr<C>& A, const C* b, const double* sigma, int S, double tol,
        int max_iter, int stop_rule, C* x, int* iterations, int* conv_iter,
        double* relres, C* r_out, double* zeta_out, double* hist, int hist_cap,
        const double* tol_scale = 0) {
    const int64_t n = A.n;
    if (S < 1 || n < 0 || max_iter < 0) return ST_EINVAL;
    std::vector<C> r(b, b + n), p(b, b + n), q(n);           // l.9-10: r <- b, p <- b
    std::vector<C> pk((size_t)S * n);
    for (int k = 0; k < S; ++k)
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) { pk[(size_t)k * n + i] = b[i]; x[(size_t)k * n + i] = C(0); }  // l.11-12
    double alpha = 0.0, beta_prev = 1.0;                      // l.2, l.4
    std::vector<double> zeta_prev(S, 1.0), zeta(S, 1.0), zeta_new(S, 1.0), beta_k(S, 0.0), alpha_k(S, 0.0);
    std::vector<char> active(S, 1);
    double R1 = dot(n, r.data(), r.data()).real();           // l.13
    const double bnorm = std::sqrt(R1);
    int it = 0, status = ST_OK, nactive = S;
    for (int k = 0; k < S; ++k) { if (conv_iter) conv_iter[k] = -1; }
    if (bnorm == 0.0) {                                       // b = 0: x_k = 0 is exact
        for (int k = 0; k < S; ++k) { if (conv_iter) conv_iter[k] = 0; if (relres) relres[k] = 0.0; if (zeta_out) zeta_out[k] = 1.0; }
        if (r_out) std::memcpy((void*)r_out, (const void*)r.data(), sizeof(C) * n);
        *iterations = 0;
        return ST_OK;
    }
    while (nactive > 0 && it < max_iter) {                    // l.15
        const double R0 = R1;                                 // l.16
        spmv(A, p.data(), q.data());                          // l.18
        const double P = dot(n, p.data(), q.data()).real();   // l.19  (Hermitian A: Im = 0, R9)
        if (!(P > 0.0) || !finite(P)) { status = ST_BREAKDOWN; break; }
        const double beta = -R0 / P;                          // l.20  (R2)
        for (int k = 0; k < S; ++k) if (active[k]) {
            const double den = beta * alpha * (zeta_prev[k] - zeta[k])
                             + zeta_prev[k] * beta_prev * (1.0 - sigma[k] * beta);
            zeta_new[k] = zeta[k] * zeta_prev[k] * beta_prev / den;     // l.22 (R3)
            beta_k[k] = beta * zeta_new[k] / zeta[k];                   // l.23 (R4)
            if (den == 0.0 || !finite(zeta_new[k]) || !finite(beta_k[k])) status = ST_BREAKDOWN;
        }
        if (status == ST_BREAKDOWN) break;
        { const C bt = rnd<C>(beta);
#pragma omp parallel for schedule(static)
          for (int64_t i = 0; i < n; ++i) r[i] = r[i] + bt * q[i]; }   // l.21
        R1 = dot(n, r.data(), r.data()).real();               // l.24
        const double alpha_next = R1 / R0;                    // l.25
        for (int k = 0; k < S; ++k) if (active[k]) {
            const double ratio = zeta_new[k] / zeta[k];
            alpha_k[k] = alpha_next * ratio * ratio;          // l.26 (R5)
        }
        { const C an = rnd<C>(alpha_next);
#pragma omp parallel for schedule(static)
          for (int64_t i = 0; i < n; ++i) p[i] = r[i] + an * p[i]; }   // l.27
        for (int k = 0; k < S; ++k) if (active[k]) {
            C* xk = x + (size_t)k * n; C* pkk = pk.data() + (size_t)k * n;
            const C bk = rnd<C>(beta_k[k]), zn = rnd<C>(zeta_new[k]), ak = rnd<C>(alpha_k[k]);
#pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < n; ++i) xk[i] = xk[i] - bk * pkk[i];            // l.28
#pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < n; ++i) pkk[i] = zn * r[i] + ak * pkk[i];       // l.29 (R6)
        }
        if (hist && it < hist_cap) {
            double* h = hist + (size_t)it * (3 + 3 * S);
            h[0] = beta; h[1] = alpha_next; h[2] = R1;
            for (int k = 0; k < S; ++k) { h[3 + k] = zeta_new[k]; h[3 + S + k] = beta_k[k]; h[3 + 2 * S + k] = alpha_k[k]; }
        }
        for (int k = 0; k < S; ++k) if (active[k]) { zeta_prev[k] = zeta[k]; zeta[k] = zeta_new[k]; }  // l.30-31
        beta_prev = beta; alpha = alpha_next; ++it;           // l.17, l.32
        const double rnorm = std::sqrt(R1);
        if (stop_rule == 1) {                                 // literal |r| > eps on the base system
            if (rnorm <= tol * bnorm) { for (int k = 0; k < S; ++k) if (active[k]) { active[k] = 0; if (conv_iter) conv_iter[k] = it; } nactive = 0; }
        } else {
            // tol_scale (multirhs only, else 1): the threshold of shift k is tol * ||b_k|| with ||b_k|| = bnorm * tol_scale[k]
            for (int k = 0; k < S; ++k) if (active[k] && std::fabs(zeta[k]) * rnorm <= tol * (bnorm * (tol_scale ? tol_scale[k] : 1.0))) {
                active[k] = 0; --nactive; if (conv_iter) conv_iter[k] = it;
                if (relres) relres[k] = std::fabs(zeta[k]) * rnorm / (bnorm * (tol_scale ? tol_scale[k] : 1.0));
            }
        }
    }
    const double rnorm = std::sqrt(R1);
    for (int k = 0; k < S; ++k) {
        if ((active[k] || stop_rule == 1) && relres) relres[k] = std::fabs(zeta[k]) * rnorm / (bnorm * (tol_scale ? tol_scale[k] : 1.0));
        if (zeta_out) zeta_out[k] = zeta[k];
    }
    if (r_out) std::memcpy((void*)r_out, (const void*)r.data(), sizeof(C) * n);
    *iterations = it;
    if (status == ST_BREAKDOWN) return status;
    return nactive > 0 ? ST_MAXITER : ST_OK;
}

// ------------------------------------------------------------------------------------------
// BiCGStab-M.  Shadow vector r0 = b.
// Shifted residual is zeta_k rho_k r.  zeta_out holds (Re, Im) of zeta_k*rho_k per shift.
// hist rows: 8+6S doubles: beta(2) chi(2) alpha_new(2) |r|^2 delta-unused, then zeta_new,
// beta_k, chi_k (complex each).
// ------------------------------------------------------------------------------------------
template <typename C>
int bicgstabm(const Csr<C>& A, const C* b, const double* sigma, int S, double tol,
              int max_iter, int stop_rule, C* x, int* iterations, int* conv_iter,
              double* relres, C* r_out, double* zeta_out, double* hist, int hist_cap,
              const double* tol_scale = 0) {
    const int64_t n = A.n;
    if (S < 1 || n < 0 || max_iter < 0) return ST_EINVAL;
    std::vector<C> r(b, b + n), p(b, b + n), r0(b, b + n), q(n), s(n), t(n), rnew(n);
    std::vector<C> pk((size_t)S * n);
    for (int k = 0; k < S; ++k)
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) { pk[(size_t)k * n + i] = b[i]; x[(size_t)k * n + i] = C(0); }
    zdouble alpha(0, 0), beta_prev(1, 0);
    std::vector<zdouble> zeta_prev(S, 1.0), zeta(S, 1.0), zeta_new(S, 1.0), rho(S, 1.0), rho_new(S, 1.0),
        beta_k(S), alpha_k(S), chi_k(S);
    std::vector<char> active(S, 1);
    zdouble delta = dot(n, r0.data(), r.data());
    double rr = delta.real();
    const double bnorm = std::sqrt(rr);
    int it = 0, status = ST_OK, nactive = S;
    for (int k = 0; k < S; ++k) { if (conv_iter) conv_iter[k] = -1; }
    if (bnorm == 0.0) {
        for (int k = 0; k < S; ++k) { if (conv_iter) conv_iter[k] = 0; if (relres) relres[k] = 0.0; if (zeta_out) { zeta_out[2 * k] = 1.0; zeta_out[2 * k + 1] = 0.0; } }
        if (r_out) std::memcpy((void*)r_out, (const void*)r.data(), sizeof(C) * n);
        *iterations = 0;
        return ST_OK;
    }
    while (nactive > 0 && it < max_iter) {
        spmv(A, p.data(), q.data());                                       // q = A p
        const zdouble r0q = dot(n, r0.data(), q.data());
        if (r0q == zdouble(0, 0) || delta == zdouble(0, 0) || !finite(r0q)) { status = ST_BREAKDOWN; break; }
        const zdouble beta = -delta / r0q;                                  // beta = -delta/<r0,q>
        for (int k = 0; k < S; ++k) if (active[k]) {
            const zdouble den = beta * alpha * (zeta_prev[k] - zeta[k])
                              + zeta_prev[k] * beta_prev * (1.0 - sigma[k] * beta);
            zeta_new[k] = zeta[k] * zeta_prev[k] * beta_prev / den;
            beta_k[k] = beta * zeta_new[k] / zeta[k];
            if (den == zdouble(0, 0) || !finite(zeta_new[k]) || !finite(beta_k[k])) status = ST_BREAKDOWN;
        }
        if (status == ST_BREAKDOWN) break;
        { const C bt = rnd<C>(beta);
#pragma omp parallel for schedule(static)
          for (int64_t i = 0; i < n; ++i) s[i] = r[i] + bt * q[i]; }       // s = r + beta q
        spmv(A, s.data(), t.data());                                       // t = A s
        const zdouble ts = dot(n, t.data(), s.data());
        const double tt = dot(n, t.data(), t.data()).real();
        if (!(tt > 0.0) || !finite(tt) || !finite(ts)) { status = ST_BREAKDOWN; break; }
        const zdouble chi = ts / tt;                                        // chi = <t,s>/<t,t>
        if (chi == zdouble(0, 0)) { status = ST_BREAKDOWN; break; }
        for (int k = 0; k < S; ++k) if (active[k]) {
            const zdouble one_cs = 1.0 + chi * sigma[k];
            if (one_cs == zdouble(0, 0)) { status = ST_BREAKDOWN; break; }
            chi_k[k] = chi / one_cs;                                        // chi_k = chi/(1+chi sigma)
            rho_new[k] = rho[k] / one_cs;                                   // rho'_k = rho_k/(1+chi sigma)
        }
        if (status == ST_BREAKDOWN) break;
        { const C ch = rnd<C>(chi);
#pragma omp parallel for schedule(static)
          for (int64_t i = 0; i < n; ++i) rnew[i] = s[i] - ch * t[i]; }    // r' = s - chi t
        const zdouble delta_new = dot(n, r0.data(), rnew.data());           // delta' = <r0,r'>
        const zdouble alpha_new = -beta * delta_new / (delta * chi);        // alpha' = -beta delta'/(delta chi)
        if (!finite(alpha_new)) { status = ST_BREAKDOWN; break; }
        for (int k = 0; k < S; ++k) if (active[k]) {
            const zdouble ratio = zeta_new[k] / zeta[k];
            alpha_k[k] = alpha_new * ratio * ratio;
        }
        for (int k = 0; k < S; ++k) if (active[k]) {
            C* xk = x + (size_t)k * n; C* pkk = pk.data() + (size_t)k * n;
            const C bk = rnd<C>(beta_k[k]);
            const C cs = rnd<C>(chi_k[k] * rho[k] * zeta_new[k]);           // coefficient of s in x_k
            const C zr = rnd<C>(zeta_new[k] * rho_new[k]);                  // coefficient of r' in p_k
            const C ak = rnd<C>(alpha_k[k]);
            const C cb = rnd<C>(chi_k[k] / beta_k[k]);
            const C zs = rnd<C>(zeta_new[k] * rho[k]);                      // s^sigma = zs * s
            const C zo = rnd<C>(zeta[k] * rho[k]);                          // r^sigma = zo * r
#pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < n; ++i) xk[i] = (xk[i] - bk * pkk[i]) + cs * s[i];
#pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < n; ++i)
                pkk[i] = zr * rnew[i] + ak * (pkk[i] - cb * (zs * s[i] - zo * r[i]));
        }
        { const C an = rnd<C>(alpha_new), ch = rnd<C>(chi);
#pragma omp parallel for schedule(static)
          for (int64_t i = 0; i < n; ++i) p[i] = rnew[i] + an * (p[i] - ch * q[i]); }  // p = r' + alpha'(p - chi q)
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) r[i] = rnew[i];
        rr = dot(n, r.data(), r.data()).real();
        if (hist && it < hist_cap) {
            double* h = hist + (size_t)it * (8 + 6 * S);
            h[0] = beta.real(); h[1] = beta.imag(); h[2] = chi.real(); h[3] = chi.imag();
            h[4] = alpha_new.real(); h[5] = alpha_new.imag(); h[6] = rr; h[7] = 0.0;
            for (int k = 0; k < S; ++k) {
                h[8 + 2 * k] = zeta_new[k].real(); h[8 + 2 * k + 1] = zeta_new[k].imag();
                h[8 + 2 * S + 2 * k] = beta_k[k].real(); h[8 + 2 * S + 2 * k + 1] = beta_k[k].imag();
                h[8 + 4 * S + 2 * k] = chi_k[k].real(); h[8 + 4 * S + 2 * k + 1] = chi_k[k].imag();
            }
        }
        for (int k = 0; k < S; ++k) if (active[k]) { zeta_prev[k] = zeta[k]; zeta[k] = zeta_new[k]; rho[k] = rho_new[k]; }
        delta = delta_new; alpha = alpha_new; beta_prev = beta; ++it;
        const double rnorm = std::sqrt(rr);
        if (!finite(rr)) { status = ST_BREAKDOWN; break; }
        if (stop_rule == 1) {
            if (rnorm <= tol * bnorm) { for (int k = 0; k < S; ++k) if (active[k]) { active[k] = 0; if (conv_iter) conv_iter[k] = it; } nactive = 0; }
        } else {
            for (int k = 0; k < S; ++k) if (active[k] && std::abs(zeta[k] * rho[k]) * rnorm <= tol * (bnorm * (tol_scale ? tol_scale[k] : 1.0))) {
                active[k] = 0; --nactive; if (conv_iter) conv_iter[k] = it;
                if (relres) relres[k] = std::abs(zeta[k] * rho[k]) * rnorm / (bnorm * (tol_scale ? tol_scale[k] : 1.0));
            }
        }
    }
    const double rnorm = std::sqrt(rr);
    for (int k = 0; k < S; ++k) {
        if ((active[k] || stop_rule == 1) && relres) relres[k] = std::abs(zeta[k] * rho[k]) * rnorm / (bnorm * (tol_scale ? tol_scale[k] : 1.0));
        if (zeta_out) { const zdouble z = zeta[k] * rho[k]; zeta_out[2 * k] = z.real(); zeta_out[2 * k + 1] = z.imag(); }
    }
    if (r_out) std::memcpy((void*)r_out, (const void*)r.data(), sizeof(C) * n);
    *iterations = it;
    if (status == ST_BREAKDOWN) return status;
    return nactive > 0 ? ST_MAXITER : ST_OK;
}

// ------------------------------------------------------------------------------------------
// A different right-hand side per shift, eq. (6):  (A + sigma_i I) x_i = b_i.
// The paper only states that "a judicious choice of initial guesses can deliver the same initial residual for
// each of the linear systems" and that generating them "involves a number of SpMV operations" ([18] is not
// available); DESIGN.md "Per-shift right-hand sides" derives the construction used here (S - 1 SpMVs):
//   Let G(s) be the vector polynomial of degree S-1 in the SHIFT variable s with G(sigma_i) = b_i, in Newton
//   form G(s) = sum_m d_m w_m(s), w_m(s) = prod_{j<m} (s - sigma_j), d_m = divided differences of the b_i.
//   Seek Y(s) = sum_{m<=S-2} u_m w_m(s) and a constant vector r0 with (A + s) Y(s) + r0 = G(s) for all s.
//   Since (A + s) w_m u_m = w_m (A + sigma_m) u_m + w_{m+1} u_m, matching the coefficients of w_m gives
//       u_{S-2} = d_{S-1};   u_{m-1} = d_m - (A + sigma_m) u_m  (m = S-2 .. 1);   r0 = d_0 - (A + sigma_0) u_0.
//   Then y_i = Y(sigma_i) = sum_{m<=i} w_m(sigma_i) u_m satisfies b_i - (A + sigma_i) y_i = r0 for EVERY i,
//   so one multishift solve (A + sigma_i) z_i = r0 from z_i = 0 finishes the family: x_i = y_i + z_i, and the
//   residual of system i is the multishift recurrence residual zeta_i r.
// Stop rule: |zeta_i| ||r|| <= tol ||b_i||  (each system relative to its own right-hand side).
// Needs pairwise distinct shifts (divided differences).  alg: 0 = CG-M, 1 = BiCGStab-M.
// y_out (S x n) and r0_out (n) are optional outputs for the pins.
// ------------------------------------------------------------------------------------------
template <typename C>
int multirhs(const Csr<C>& A, const C* B, const double* sigma, int S, double tol, int max_iter, int alg,
             C* x, int* iterations, int* conv_iter, double* relres, C* y_out, C* r0_out) {
    const int64_t n = A.n;
    if (S < 1 || n < 0 || max_iter < 0) return ST_EINVAL;
    for (int i = 0; i < S; ++i)
        for (int j = 0; j < i; ++j) if (sigma[i] == sigma[j]) return ST_EINVAL;
    // ||b_i||
    std::vector<double> bn(S);
    for (int i = 0; i < S; ++i) bn[i] = std::sqrt(dot(n, B + (size_t)i * n, B + (size_t)i * n).real());
    // divided differences, in place: after level l, D[i] = b[sigma_{i-l}, ..., sigma_i] for i >= l
    std::vector<C> D(B, B + (size_t)S * n);
    for (int l = 1; l < S; ++l)
        for (int i = S - 1; i >= l; --i) {
            const C inv = rnd<C>(1.0 / (sigma[i] - sigma[i - l]));
            C* di = D.data() + (size_t)i * n; const C* dm = D.data() + (size_t)(i - 1) * n;
            for (int64_t e = 0; e < n; ++e) di[e] = (di[e] - dm[e]) * inv;
        }
    // u recursion, in place: slot m+1 holds u_m, slot 0 ends as r0
    std::vector<C> q(n);
    for (int m = S - 2; m >= 0; --m) {
        const C* um = D.data() + (size_t)(m + 1) * n;
        C* dst = D.data() + (size_t)m * n;
        spmv(A, um, q.data());
        const C sg = rnd<C>(sigma[m]);
        for (int64_t e = 0; e < n; ++e) dst[e] = dst[e] - (q[e] + sg * um[e]);
    }
    const C* r0 = D.data();
    if (r0_out) std::memcpy((void*)r0_out, (const void*)r0, sizeof(C) * n);
    const double r0n = std::sqrt(dot(n, r0, r0).real());
    // (A + sigma_i) z_i = r0 from z_i = 0, thresholds tol ||b_i||
    std::vector<double> ts(S);
    for (int i = 0; i < S; ++i) ts[i] = r0n > 0.0 ? bn[i] / r0n : 1.0;
    int status;
    if (alg == 0) status = cgm(A, r0, sigma, S, tol, max_iter, 0, x, iterations, conv_iter, relres, (C*)0, (double*)0, (double*)0, 0, ts.data());
    else status = bicgstabm(A, r0, sigma, S, tol, max_iter, 0, x, iterations, conv_iter, relres, (C*)0, (double*)0, (double*)0, 0, ts.data());
    // x_i = z_i + y_i,  y_i = sum_{m <= min(i, S-2)} w_m(sigma_i) u_m
    for (int i = 0; i < S; ++i) {
        C* xi = x + (size_t)i * n;
        C* yi = y_out ? y_out + (size_t)i * n : (C*)0;
        if (yi) for (int64_t e = 0; e < n; ++e) yi[e] = C(0);
        double w = 1.0;
        for (int m = 0; m <= i && m <= S - 2; ++m) {
            const C wc = rnd<C>(w);
            const C* um = D.data() + (size_t)(m + 1) * n;
            for (int64_t e = 0; e < n; ++e) xi[e] = xi[e] + wc * um[e];
            if (yi) for (int64_t e = 0; e < n; ++e) yi[e] = yi[e] + wc * um[e];
            w *= sigma[i] - sigma[m];
        }
    }
    return status;
}

// ------------------------------------------------------------------------------------------
// Plain CG on (A + sigma I), textbook form ([13]).  Pin only.
// ------------------------------------------------------------------------------------------
template <typename C>
int cg(const Csr<C>& A, double sigma, const C* b, double tol, int max_iter,
       C* x, int* iterations, double* relres) {
    const int64_t n = A.n;
    std::vector<C> r(b, b + n), p(b, b + n), q(n);
    for (int64_t i = 0; i < n; ++i) x[i] = C(0);
    double rr = dot(n, r.data(), r.data()).real();
    const double bnorm = std::sqrt(rr);
    int it = 0, status = ST_MAXITER;
    if (bnorm == 0.0) { *iterations = 0; if (relres) *relres = 0.0; return ST_OK; }
    while (it < max_iter) {
        spmv(A, p.data(), q.data());
        if (sigma != 0.0) { const C sg = rnd<C>(sigma); for (int64_t i = 0; i < n; ++i) q[i] = q[i] + sg * p[i]; }
        const double pq = dot(n, p.data(), q.data()).real();
        if (!(pq > 0.0)) { status = ST_BREAKDOWN; break; }
        const double a = rr / pq;
        const C ac = rnd<C>(a);
        for (int64_t i = 0; i < n; ++i) x[i] = x[i] + ac * p[i];
        for (int64_t i = 0; i < n; ++i) r[i] = r[i] - ac * q[i];
        const double rr_new = dot(n, r.data(), r.data()).real();
        const double bt = rr_new / rr;
        const C bc = rnd<C>(bt);
        for (int64_t i = 0; i < n; ++i) p[i] = r[i] + bc * p[i];
        rr = rr_new; ++it;
        if (std::sqrt(rr) <= tol * bnorm) { status = ST_OK; break; }
    }
    *iterations = it;
    if (relres) *relres = std::sqrt(rr) / bnorm;
    return status;
}

// ------------------------------------------------------------------------------------------
// Plain BiCGStab on (A + sigma I), van der Vorst's form, shadow vector b.  Pin only.
// ------------------------------------------------------------------------------------------
template <typename C>
int bicgstab(const Csr<C>& A, double sigma, const C* b, double tol, int max_iter,
             C* x, int* iterations, double* relres) {
    const int64_t n = A.n;
    std::vector<C> r(b, b + n), p(b, b + n), rhat(b, b + n), v(n), s(n), t(n);
    for (int64_t i = 0; i < n; ++i) x[i] = C(0);
    zdouble rho = dot(n, rhat.data(), r.data());
    double rr = rho.real();
    const double bnorm = std::sqrt(rr);
    int it = 0, status = ST_MAXITER;
    if (bnorm == 0.0) { *iterations = 0; if (relres) *relres = 0.0; return ST_OK; }
    const C sg = rnd<C>(sigma);
    while (it < max_iter) {
        spmv(A, p.data(), v.data());
        if (sigma != 0.0) for (int64_t i = 0; i < n; ++i) v[i] = v[i] + sg * p[i];
        const zdouble rv = dot(n, rhat.data(), v.data());
        if (rv == zdouble(0, 0) || rho == zdouble(0, 0)) { status = ST_BREAKDOWN; break; }
        const zdouble a = rho / rv;
        const C ac = rnd<C>(a);
        for (int64_t i = 0; i < n; ++i) s[i] = r[i] - ac * v[i];
        spmv(A, s.data(), t.data());
        if (sigma != 0.0) for (int64_t i = 0; i < n; ++i) t[i] = t[i] + sg * s[i];
        const zdouble ts = dot(n, t.data(), s.data());
        const double tt = dot(n, t.data(), t.data()).real();
        if (!(tt > 0.0)) { status = ST_BREAKDOWN; break; }
        const zdouble w = ts / tt;
        const C wc = rnd<C>(w);
        for (int64_t i = 0; i < n; ++i) x[i] = (x[i] + ac * p[i]) + wc * s[i];
        for (int64_t i = 0; i < n; ++i) r[i] = s[i] - wc * t[i];
        const zdouble rho_new = dot(n, rhat.data(), r.data());
        const zdouble bt = (rho_new / rho) * (a / w);
        const C bc = rnd<C>(bt);
        for (int64_t i = 0; i < n; ++i) p[i] = r[i] + bc * (p[i] - wc * v[i]);
        rho = rho_new; ++it;
        rr = dot(n, r.data(), r.data()).real();
        if (std::sqrt(rr) <= tol * bnorm) { status = ST_OK; break; }
    }
    *iterations = it;
    if (relres) *relres = std::sqrt(rr) / bnorm;
    return status;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// C entry points (host pointers only).
// dtype: 0 = complex64, 1 = complex128, 2 = float32, 3 = float64 (real: the paper's Table 1 runs).
// ------------------------------------------------------------------------------------------
typedef std::complex<float> cfloat;

template <typename C>
static Csr<C> mk(int64_t n, const int32_t* rp, const int32_t* ci, const void* v) {
    Csr<C> A; A.n = n; A.rowptr = rp; A.colidx = ci; A.val = (const C*)v; return A;
}

#define DISPATCH(F, ...)                                  \
    switch (dtype) {                                      \
        case 0: return F<cfloat>(__VA_ARGS__);            \
        case 1: return F<zdouble>(__VA_ARGS__);           \
        case 2: return F<float>(__VA_ARGS__);             \
        case 3: return F<double>(__VA_ARGS__);            \
        default: return (int)ST_EINVAL;                   \
    }

template <typename C>
static int spmv_entry(int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val, const void* x, void* y) {
    spmv(mk<C>(n, rowptr, colidx, val), (const C*)x, (C*)y);
    return 0;
}
template <typename C>
static int cgm_entry(int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val, const void* b,
                     const double* shifts, int nshifts, double tol, int max_iter, int stop_rule, void* x,
                     int* iterations, int* conv_iter, double* relres, void* r_out, double* zeta_out, double* hist, int hist_cap) {
    return cgm(mk<C>(n, rowptr, colidx, val), (const C*)b, shifts, nshifts, tol, max_iter, stop_rule, (C*)x,
               iterations, conv_iter, relres, (C*)r_out, zeta_out, hist, hist_cap);
}
template <typename C>
static int bicgstabm_entry(int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val, const void* b,
                           const double* shifts, int nshifts, double tol, int max_iter, int stop_rule, void* x,
                           int* iterations, int* conv_iter, double* relres, void* r_out, double* zeta_out, double* hist, int hist_cap) {
    return bicgstabm(mk<C>(n, rowptr, colidx, val), (const C*)b, shifts, nshifts, tol, max_iter, stop_rule, (C*)x,
                     iterations, conv_iter, relres, (C*)r_out, zeta_out, hist, hist_cap);
}
template <typename C>
static int multirhs_entry(int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val, const void* B,
                          const double* shifts, int nshifts, double tol, int max_iter, int alg, void* x,
                          int* iterations, int* conv_iter, double* relres, void* y_out, void* r0_out) {
    return multirhs(mk<C>(n, rowptr, colidx, val), (const C*)B, shifts, nshifts, tol, max_iter, alg, (C*)x,
                    iterations, conv_iter, relres, (C*)y_out, (C*)r0_out);
}
template <typename C>
static int cg_entry(int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val, double sigma,
                    const void* b, double tol, int max_iter, void* x, int* iterations, double* relres) {
    return cg(mk<C>(n, rowptr, colidx, val), sigma, (const C*)b, tol, max_iter, (C*)x, iterations, relres);
}
template <typename C>
static int bicgstab_entry(int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val, double sigma,
                          const void* b, double tol, int max_iter, void* x, int* iterations, double* relres) {
    return bicgstab(mk<C>(n, rowptr, colidx, val), sigma, (const C*)b, tol, max_iter, (C*)x, iterations, relres);
}

extern "C" {

int oracle_spmv_csr(int dtype, int64_t n, const int32_t* rowptr, const int32_t* colidx,
                    const void* val, const void* x, void* y) {
    DISPATCH(spmv_entry, n, rowptr, colidx, val, x, y)
}

int oracle_cgm(int dtype, int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val,
               const void* b, const double* shifts, int nshifts, double tol, int max_iter, int stop_rule,
               void* x, int* iterations, int* conv_iter, double* relres,
               void* r_out, double* zeta_out, double* hist, int hist_cap) {
    DISPATCH(cgm_entry, n, rowptr, colidx, val, b, shifts, nshifts, tol, max_iter, stop_rule, x, iterations,
             conv_iter, relres, r_out, zeta_out, hist, hist_cap)
}

int oracle_bicgstabm(int dtype, int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val,
                     const void* b, const double* shifts, int nshifts, double tol, int max_iter, int stop_rule,
                     void* x, int* iterations, int* conv_iter, double* relres,
                     void* r_out, double* zeta_out, double* hist, int hist_cap) {
    DISPATCH(bicgstabm_entry, n, rowptr, colidx, val, b, shifts, nshifts, tol, max_iter, stop_rule, x, iterations,
             conv_iter, relres, r_out, zeta_out, hist, hist_cap)
}

int oracle_multirhs(int dtype, int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val,
                    const void* B, const double* shifts, int nshifts, double tol, int max_iter, int alg,
                    void* x, int* iterations, int* conv_iter, double* relres, void* y_out, void* r0_out) {
    DISPATCH(multirhs_entry, n, rowptr, colidx, val, B, shifts, nshifts, tol, max_iter, alg, x, iterations,
             conv_iter, relres, y_out, r0_out)
}

int oracle_cg(int dtype, int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val,
              double sigma, const void* b, double tol, int max_iter, void* x, int* iterations, double* relres) {
    DISPATCH(cg_entry, n, rowptr, colidx, val, sigma, b, tol, max_iter, x, iterations, relres)
}

int oracle_bicgstab(int dtype, int64_t n, const int32_t* rowptr, const int32_t* colidx, const void* val,
                    double sigma, const void* b, double tol, int max_iter, void* x, int* iterations, double* relres) {
    DISPATCH(bicgstab_entry, n, rowptr, colidx, val, sigma, b, tol, max_iter, x, iterations, relres)
}

}  // extern "C"
