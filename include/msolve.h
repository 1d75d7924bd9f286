/* msolve.h -- C ABI of the B200-native multishift Krylov solvers CG-M and BiCGStab-M.
 *
 * The library solves the family of shifted systems of eq. (1), PAPER.md:41,
 *
 *        (A + sigma_k I) x_k = b ,   k = 0 .. nshifts-1 ,
 *
 * for all shifts from ONE Krylov sequence (eq. (4)): CG-M is Algorithm 1
 * for Hermitian positive-definite A, BiCGStab-M is its
 * non-Hermitian analogue.  The argument lists follow the paper's statement of the problem and
 * the call of Fig. 1: a sparse A, a right-hand side b of length n, an array
 * of shifts, a relative tolerance and an iteration limit (the paper's
 * `default_monitor(b, 2000, 1e-5)`) and ONE output array of n*nshifts holding one
 * solution per shift.  The initial guess is zero by construction of the method
 * (PAPER.md:97, 232).
 *
 * Everything on the iteration path runs in hand-written sm_100a kernels; the whole iteration
 * is captured in a CUDA graph and loops on the device without host synchronisation
 * (the paper's "entire solution on the GPU").
 *
 * Conventions
 *  - Plain C, no exceptions.  Every int-returning call returns an MSOLVE_* status code;
 *    msolve_last_error() gives the text of the last failure of the calling thread.
 *  - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  Device buffers are owned
 *    by the caller (e.g. torch tensors); the library never frees them.
 *  - Elements are interleaved (re, im) pairs of float (MSOLVE_C64) or double (MSOLVE_C128), or
 *    plain float / double (MSOLVE_F32 / MSOLVE_F64).  "complex" below means "element of the
 *    handle's dtype".  Indices are int32.  All device arrays must be 16-byte aligned.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *  - A handle may be used by one solve at a time (it owns the device-side solver state and the
 *    cached CUDA graphs); different handles are independent.  A handle belongs to the device that
 *    was current when it was created; calls made with another current device return MSOLVE_EINVAL.
 */
#ifndef MSOLVE_H
#define MSOLVE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct msolve_matrix msolve_matrix; /* opaque */

/* Element type of the matrix and of every vector.  Complex = interleaved (re, im) pairs: the
 * BASELINE lattice / unstructured configs.  Real: the paper's own measurements are real fp32 /
 * fp64 (Table 1); CSR only. */
enum { MSOLVE_C64 = 0, MSOLVE_C128 = 1, MSOLVE_F32 = 2, MSOLVE_F64 = 3 };

enum { MSOLVE_ALG_CGM = 0, MSOLVE_ALG_BICGSTABM = 1 };

/* Status codes.  > 0: x is valid but the solve did not end with every shift converged. */
enum {
    MSOLVE_OK = 0,         /* every shift reached |zeta_k| ||r|| <= tol ||b||                      */
    MSOLVE_MAXITER = 1,    /* iteration limit reached first                                        */
    MSOLVE_BREAKDOWN = 2,  /* <p,Ap> <= 0, <r0,Ap> = 0, <t,t> = 0, zero zeta denominator, NaN/Inf */
    MSOLVE_EINVAL = -1,    /* bad argument (nothing was launched)                                  */
    MSOLVE_ECUDA = -2,     /* a CUDA call failed; see msolve_last_error()                          */
    MSOLVE_ENOMEM = -3     /* workspace too small / allocation failed                              */
};

/* create-time flags: SpMV kernel choice for CSR (Alg. 1 l.18). */
enum {
    MSOLVE_SPMV_AUTO = 0,    /* TMA-staged vector-CSR for short rows, else vector or merge-path */
    MSOLVE_SPMV_VECTOR = 1,  /* sub-warp-per-row vector-CSR                                 */
    MSOLVE_SPMV_MERGE = 2,   /* merge-path CSR (load-balanced over rows + non-zeros)        */
    MSOLVE_SPMV_TILE = 3     /* TMA-staged vector-CSR (rows of at most 64 non-zeros for 16-byte elements, 128 otherwise) */
};

#define MSOLVE_MAX_SHIFTS 128

/* msolve_config keys (per handle) */
enum {
    MSOLVE_CFG_LOOP_MODE = 0, /* 0 = device WHILE graph node (default), 1 = chunked relaunch of an
                                 unrolled iteration graph with a device `done` flag */
    MSOLVE_CFG_UPDATE_KERNEL = 1 /* CG-M fused multishift update: 0 = register kernel (default), 1 = TMA-staged
                                    kernel (bulk async loads AND stores) whenever the vector length is a multiple
                                    of 16 bytes.  Same arithmetic; both run at the same 6.0 TB/s on B200 */,
    MSOLVE_CFG_LATTICE_KERNEL = 2 /* tile kernel of msolve_create_lattice_su3 handles: 0 = the fastest one for the
                                     lattice and element type (default: 4 where it applies, else 3 for complex128 and
                                     2 for complex64), 1 = (term, site) threads + partials, 2 = warp per tile,
                                     3 = hybrid (forward links by bulk copy, backward links and neighbours gathered),
                                     4 = blocked (a tile is a block of x0-rows in the (x1, x2) plane whose interior
                                     neighbours are staged once; 4-D lattices with L0 = 32 whose extents the block
                                     divides, any other handle takes the default instead) */,
    MSOLVE_CFG_STOP_RULE = 3 /* 0 = per shift (default): shift k stops, and x_k is frozen, at the first iteration with
                                |zeta_k| ||r|| <= tol ||b|| (the paper is silent on masking; R15).
                                1 = Alg. 1 l.15 read literally ("while |r| > eps"): every shift keeps
                                iterating until the residual of the UNSHIFTED system has ||r|| <= tol ||b||, then all
                                stop together (conv_iter[k] = that iteration for every k) */,
    MSOLVE_CFG_X_WINDOW = 4 /* vector-CSR kernel only: 1 = every SpMV launch carries an L2 access-policy window over the
                               gathered vector (persisting hits; sets the device-wide persisting-L2 set-aside).
                               Measured on B200, config 5: profiles/r02_sweeps.md; default 0 */,
    MSOLVE_CFG_MATRIX_L2 = 5 /* L2 policy of the matrix stream of the TMA-staged SpMV kernels: 0 / 1 = evict-first (default:
                                the matrix is read once per SpMV), 2 = evict-last.  Keeping a matrix that fits in L2
                                (config 3: 88 MB of 126 MB) was measured and is slower: 11.4k -> 9.9k iterations/s
                                (profiles/r02_sweeps.md); the option stays for that measurement */,
    MSOLVE_CFG_ITER_PATH = 6 /* how a solve is driven: 1 = the iteration as a CUDA graph of kernels looping on the device
                                (one kernel per step of Alg. 1; HBM-bound sizes), 2 = the WHOLE solve as one cooperative
                                kernel with grid-wide barriers between the steps (systems that live in L2, where kernel
                                launches, not bytes, are the cost; vector-CSR, BSR3 and lattice handles), 3 = one
                                cooperative kernel with the matrix and every vector RESIDENT IN SHARED MEMORY (CSR / BSR3
                                handles whose matrix and 3 + 2 nshifts (BiCGStab-M: 6 + 2 nshifts) vectors fit in the
                                shared memory of the SMs, a few MB: only the gathered vector and the dot products touch
                                global memory per iteration),
                                0 = by footprint (default): 3 when it fits, else 2 when matrix + (4 + 2 nshifts) vectors
                                take at most 256 MB (96 MB for CG-M with the deferred update, whose graph of
                                kernels moves 2.2 times fewer bytes per iteration), else 1.
                                Same arithmetic step for step; the paths group the dot products differently (per-CTA
                                partials of different grids), so they agree to rounding, not bit for bit */,
    MSOLVE_CFG_FUSED_CTAS = 7 /* CTAs of the cooperative kernel of MSOLVE_CFG_ITER_PATH = 2: 0 = by problem size
                                 (default), else that many (at most one per SM) */,
    MSOLVE_CFG_MATRIX_L2_KEEP_PERCENT = 8 /* 0 .. 100: that share of the matrix stream (cache lines picked by the
                                 hardware from the address, createpolicy.fractional) is loaded evict-last, the rest
                                 evict-first -- for a matrix of which a part fits in L2 next to the vectors.  Applies to
                                 the TMA-staged kernels and to the BSR3 SpMV of the one-kernel path;
                                 MSOLVE_CFG_MATRIX_L2 = 1 / 2 set it to 0 / 100.  Default 0; profiles/r02_sweeps.md */,
    MSOLVE_CFG_DEFER_UPDATE = 9 /* CG-M as a graph of kernels: chunk length M of the DEFERRED multishift update, 0 .. 32,
                                 default 32.  Alg. 1 l.28-29 write every x_k and p_k in every
                                 iteration; both are linear in the residuals r_n with coefficients the scalar
                                 recurrences already produce, so with M > 0 an iteration only updates r (kept in a ring
                                 of M + 1 vectors) while the scalar kernel accumulates 2 M + 2 fp64 coefficients per
                                 shift, and one pass per M iterations (and one when the solve ends) forms p_k and x_k:
                                 (M + 4 nshifts) / M vector passes per iteration instead of 4 nshifts.  The scalars,
                                 residuals and stop decisions are those of M = 0 (they do not involve x_k, p_k); x_k
                                 agrees to rounding (other order of the additions).  Costs M vectors of workspace (msolve_workspace_bytes counts
                                 them).  0 = the update of every iteration.  BiCGStab-M, the one-kernel paths, the row
                                 partition and MSOLVE_CFG_UPDATE_KERNEL = 1 always run the step-by-step form */
};

/* Build a handle for a CSR matrix (n x n).  Borrows the three device arrays: they must stay
 * valid and unchanged until msolve_destroy.  Column indices must lie in [0, n).  May allocate
 * library-owned auxiliary device data (merge-path partition table, solver state).
 * flags: MSOLVE_SPMV_AUTO reads d_rowptr once at create time and takes the TMA-staged vector-CSR
 * kernel when no row is longer than MSOLVE_SPMV_TILE allows (and d_rowptr / d_colidx are 16-byte
 * aligned), merge-path when single rows dwarf the mean, the plain vector kernel otherwise; the
 * other values force one kernel (EINVAL when the matrix does not fit it).
 * Errors: EINVAL (null pointer, n < 0, nnz < 0, bad dtype/flags, nnz >= 2^31), ECUDA, ENOMEM. */
int msolve_create_csr(msolve_matrix **A, int64_t n, int64_t nnz,
                      const int32_t *d_rowptr /* n+1 */, const int32_t *d_colidx /* nnz */,
                      const void *d_val /* nnz complex */, int dtype, int flags, void *stream);

/* Build a handle for a 3x3-block BSR matrix (3*nbrows x 3*nbrows), the SU(3) layout:
 * block k is 9 complex numbers, row-major 3x3, at d_blocks + 9*k.  Same borrowing rules.
 * flags: MSOLVE_SPMV_AUTO = TMA-staged tile kernel when the rows allow it (reads d_browptr once
 * at create time to build its tile table), MSOLVE_SPMV_VECTOR = simple thread-per-row kernel. */
int msolve_create_bsr3(msolve_matrix **A, int64_t nbrows, int64_t nblocks,
                       const int32_t *d_browptr /* nbrows+1 */, const int32_t *d_bcolidx /* nblocks */,
                       const void *d_blocks /* nblocks*9 complex */, int dtype, int flags, void *stream);

/* Matrix-free handle for the gauged lattice operator with SU(3) links (the "custom linear
 * operator" hook of PAPER.md:146 applied to the operator of BASELINE configs 2-4):
 *
 *   (A x)(s) = diag x(s) - sum_mu [ c_f U_mu(s) x(s+mu) + c_b U_mu(s-mu)^dagger x(s-mu) ]
 *
 * on a periodic lattice of `ndim` (1..4) dimensions with extents h_extents[0..ndim-1] (host), site
 * index s = x0 + L0 (x1 + L1 (x2 + L2 x3)), scalar row = 3 s + colour, n = 3 V.  d_links holds
 * links[mu][s] = U_mu(s): ndim * V blocks of 9 complex, row-major 3x3 (borrowed, as above).
 * The assembled form of the same operator is what msolve_create_bsr3 takes; this handle reads 4
 * link blocks per site instead of 9 matrix blocks + indices.  dtype: MSOLVE_C64 / MSOLVE_C128.
 * flags: MSOLVE_SPMV_AUTO = TMA-staged tile kernel when an x0-row is a 16-byte multiple and at most
 * 32 sites, MSOLVE_SPMV_VECTOR = thread-per-row kernel (any extents).
 * Errors: EINVAL (ndim, extents, null / misaligned pointer, dtype, flags, 3 V >= 2^31), ECUDA. */
int msolve_create_lattice_su3(msolve_matrix **A, int ndim, const int32_t *h_extents /* ndim */,
                              const void *d_links /* ndim*V*9 complex */, double diag, double c_f,
                              double c_b, int dtype, int flags, void *stream);

/* Bytes of caller-provided device workspace a solve with `nshifts` shifts needs
 * (r, p, Ap [, s, t] and one search direction p_k per shift, Alg. 1 l.10-11; for CG-M also the MSOLVE_CFG_DEFER_UPDATE
 * residuals of the deferred update, as the handle is configured WHEN THIS IS CALLED: ask again after msolve_config).
 * 0 on bad input. */
size_t msolve_workspace_bytes(const msolve_matrix *A, int nshifts, int algorithm);

/* CG-M, Algorithm 1 as read in DESIGN.md ("Readings of the paper").
 *   d_b          in   n complex, device.  Not modified.
 *   h_shifts     in   nshifts real shifts sigma_k (host), any order, 1 <= nshifts <= MSOLVE_MAX_SHIFTS.
 *   tol          in   relative tolerance: shift k stops (and x_k is frozen) at the first iteration
 *                     with |zeta_k| ||r|| <= tol ||b||; the solve ends when all shifts stopped.
 *   max_iter     in   limit on loop bodies (one SpMV each for CG-M, two for BiCGStab-M).
 *   d_x          out  nshifts*n complex, device, shift-major: x_k[i] at d_x[k*n + i].  Fully
 *                     overwritten (zero initial guess is part of the method; a solve that stops before its
 *                     first update -- b = 0, max_iter = 0, breakdown in the first loop body -- returns x = 0).
 *   d_workspace       device scratch of >= msolve_workspace_bytes(), 256-byte aligned.
 *   h_iterations out  loop bodies executed (may be NULL).
 *   h_conv_iter  out  nshifts ints: iteration at which shift k converged, -1 if it did not (or NULL).
 *   h_relres     out  nshifts doubles: recurrence residual |zeta_k| ||r|| / ||b|| when shift k
 *                     stopped / at exit (or NULL).
 * Host outputs are written after ONE stream synchronisation at the end of the solve; there is no
 * host synchronisation per iteration.  Returns OK / MAXITER / BREAKDOWN or a negative error. */
int msolve_cgm(const msolve_matrix *A, const void *d_b, const double *h_shifts, int nshifts,
               double tol, int max_iter, void *d_x, void *d_workspace, size_t workspace_bytes,
               int *h_iterations, int *h_conv_iter, double *h_relres, void *stream);

/* BiCGStab-M (derivation in DESIGN.md), shadow vector r0 = b.  Same arguments.
 * Stop test per shift: |zeta_k rho_k| ||r|| <= tol ||b||, evaluated at the end of a full iteration. */
int msolve_bicgstabm(const msolve_matrix *A, const void *d_b, const double *h_shifts, int nshifts,
                     double tol, int max_iter, void *d_x, void *d_workspace, size_t workspace_bytes,
                     int *h_iterations, int *h_conv_iter, double *h_relres, void *stream);

/* A different right-hand side per shift, eq. (6):  (A + sigma_i I) x_i = b_i.
 * "A judicious choice of initial guesses can deliver the same initial residual for each of the linear systems"
 * (PAPER.md:232): the library builds initial guesses y_i with b_i - (A + sigma_i) y_i = r0 for every i on the
 * device (Newton divided differences of the b_i in the shift variable, nshifts - 1 SpMVs; derivation in DESIGN.md
 * "Per-shift right-hand sides"), runs ONE multishift solve (A + sigma_i) z_i = r0 with the unchanged CG-M /
 * BiCGStab-M iteration and returns x_i = y_i + z_i.
 *   d_B          in   nshifts*n complex, device, shift-major: b_i[j] at d_B[i*n + j].  Not modified.
 *   h_shifts     in   pairwise DISTINCT (EINVAL otherwise: two systems with one shift and two right-hand sides do
 *                     not share a Krylov space).
 *   tol          in   system i stops at |zeta_i| ||r|| <= tol ||b_i||: relative to ITS OWN right-hand side;
 *                     h_relres[i] is that ratio.
 *   d_workspace       >= msolve_multirhs_workspace_bytes(): the solver's workspace plus nshifts vectors.
 * Everything else as msolve_cgm.
 * Numerical range: r0 is the interpolant of the b_i over the shifts, EXTRAPOLATED to s = -spec(A).  For right-hand
 * sides that vary smoothly with the shift that is harmless; for independent ones ||r0|| / ||b|| grows like
 * ||A||^(nshifts-1) / prod |sigma_i - sigma_j|, and tol is reachable only while eps ||r0|| < tol ||b_i|| (eps of the
 * element type).  A handful of well separated shifts is the practical range (tests: 3 smooth systems in both
 * precisions, 5 independent ones in complex128, 20 for an operator that is small against the shift spacing). */
size_t msolve_multirhs_workspace_bytes(const msolve_matrix *A, int nshifts, int algorithm);
int msolve_solve_multirhs(const msolve_matrix *A, int algorithm, const void *d_B, const double *h_shifts,
                          int nshifts, double tol, int max_iter, void *d_x, void *d_workspace,
                          size_t workspace_bytes, int *h_iterations, int *h_conv_iter, double *h_relres,
                          void *stream);

/* The call of Fig. 1 with HOST vectors: copies h_b to the device, solves,
 * copies all nshifts*n solutions back to h_x (both inside the call, on `stream`).  The library
 * allocates the device vectors and workspace itself and keeps them in the handle for the next call
 * (grow-only; freed by msolve_destroy).  algorithm = MSOLVE_ALG_*. */
int msolve_solve_host(const msolve_matrix *A, int algorithm, const void *h_b, const double *h_shifts,
                      int nshifts, double tol, int max_iter, void *h_x,
                      int *h_iterations, int *h_conv_iter, double *h_relres, void *stream);

/* The same for a batch of nrhs right-hand sides of one family (RHMC solves the same shifted family for
 * several pseudofermion fields): h_b[i] -> h_x[i] (nshifts*n each, shift-major), solved one
 * after the other on `stream`, software-pipelined: the device-to-host copy of solution set i and the host-to-device
 * copy of the NEXT right-hand side run on two library-owned copy streams while a solve is running (two
 * device slots of b and x, kept in the handle).
 * Host vectors should be pinned, or the copies do not overlap.  h_iterations: nrhs; h_conv_iter,
 * h_relres: nrhs*nshifts (or NULL).  Returns the largest status of the solves (MSOLVE_OK / MAXITER /
 * BREAKDOWN) or the first error (< 0); all copies have completed on return. */
int msolve_solve_host_batch(const msolve_matrix *A, int algorithm, int nrhs, const void *const *h_b,
                            const double *h_shifts, int nshifts, double tol, int max_iter,
                            void *const *h_x, int *h_iterations, int *h_conv_iter, double *h_relres,
                            void *stream);

/* One SpMV y = A x with the fused reduction of the CG-M step (Alg. 1 l.18-19):
 * h_dot[0..1] receives <x, A x> = sum_i conj(x_i) y_i (may be NULL).  d_x, d_y: n complex, device.
 * Exposed for parity tests of the SpMV kernels and for per-kernel timing. */
int msolve_spmv(const msolve_matrix *A, const void *d_x, void *d_y, double *h_dot, void *stream);

/* The same operation for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): y = A x for a CSR matrix and d_dot[0..1] = <x, A x> = sum_i conj(x_i) y_i
 * (Alg. 1 l.18-19), without a handle.  The call allocates NOTHING (no cudaMalloc / cudaFree, no
 * allocating library routine) and does not synchronise: two kernels are enqueued on `stream`.
 *   n                 rows = columns, 0 <= n <= MSOLVE_NOALLOC_MAX_ROWS, else MSOLVE_EINVAL (nothing is launched);
 *   d_rowptr [n+1], d_colidx [nnz], d_val [nnz]: device CSR arrays, borrowed, column indices in [0, n);
 *   dtype             MSOLVE_C64 / C128 / F32 / F64: element type of d_val, d_x, d_y;
 *   d_x [n] in, d_y [n] out, d_dot [2 doubles: re, im] out: device, caller-owned, aligned to their element size;
 *                     for real types d_dot[1] = 0.  d_y must not alias d_x.
 * Scratch: one (re, im) partial per 64 rows in a static device array of MSOLVE_NOALLOC_MAX_ROWS / 64 * 16 bytes =
 * 256 KiB, which every GPU that loads the library holds until the process exits.  The first call on a device
 * resolves the array's device address (cudaGetSymbolAddress, once per device): make that call outside graph
 * capture.  All calls share the array: calls that overlap on the GPU (different streams, graph branches without a
 * dependency between them) RACE on it and must be serialised by the caller; nothing in it needs clearing between
 * calls (a call reads only the partials it has written itself).  Larger systems: msolve_create_csr + msolve_spmv.
 * Returns MSOLVE_OK / MSOLVE_EINVAL / MSOLVE_ECUDA. */
#define MSOLVE_NOALLOC_MAX_ROWS 1048576
int msolve_spmv_csr_noalloc(int64_t n, const int32_t *d_rowptr, const int32_t *d_colidx, const void *d_val, int dtype,
                            const void *d_x, void *d_y, double *d_dot, void *stream);

/* Per-kernel timing of `iters` steady-state iterations (no convergence test, all shifts active),
 * each kernel bracketed by CUDA events on `stream`.  h_ms[j] receives the mean duration in ms of
 * kernel j, h_launches[j] its launches per iteration; names via msolve_kernel_name(algorithm, j).
 * Returns the number of kernels (<= 8) or a negative error.  d_x / workspace as for the solvers. */
int msolve_profile_iteration(const msolve_matrix *A, int algorithm, const void *d_b,
                             const double *h_shifts, int nshifts, int iters, void *d_x,
                             void *d_workspace, size_t workspace_bytes,
                             float *h_ms /* 8 */, int *h_launches /* 8 */, void *stream);
const char *msolve_kernel_name(int algorithm, int j);

/* Kernel launches issued (graph kernel nodes executed) by the last solve on this handle. */
int64_t msolve_last_launch_count(const msolve_matrix *A);

/* Set option `key` (MSOLVE_CFG_*) of this handle; it holds for every later call on the handle.
 * Returns MSOLVE_OK or MSOLVE_EINVAL (NULL handle, unknown key, value out of range). */
int msolve_config(msolve_matrix *A, int key, int value);

/* Per-iteration scalar history (the quantities of Alg. 1 l.20-26, which otherwise never
 * leave the device): every later solve on this handle writes one row per completed iteration n = 0, 1, ...
 * into d_hist (device, 8-byte aligned, borrowed, at least cap_rows rows), rows beyond cap_rows are dropped.
 *   CG-M row,        3 + 3 S doubles: beta_n, alpha_{n+1}, R1 = ||r_{n+1}||^2, then zeta_{n+1,k} [S], beta_{n,k} [S],
 *                    alpha_{n+1,k} [S];
 *   BiCGStab-M row,  8 + 6 S doubles: beta (re, im), chi (re, im), alpha' (re, im), ||r'||^2, 0, then zeta_new_k [S],
 *                    beta_k [S], chi_k [S] as (re, im) pairs.
 * A shift that has stopped keeps the values of its last active iteration.  An iteration that breaks down
 * writes no row.  cap_rows = 0 (or d_hist = NULL) switches the history off.  Returns OK / EINVAL. */
int msolve_set_history(msolve_matrix *A, double *d_hist, int cap_rows);

/* Where the time of the one-kernel path (MSOLVE_CFG_ITER_PATH = 2) goes: while d_ns is set, thread 0 of CTA 0 reads
 * %globaltimer at every phase boundary of every later solve on this handle and ADDS the nanoseconds into
 * d_ns[0 .. 15] (device, uint64, 8-byte aligned, borrowed; the caller zeroes it):
 *   CG-M:        [0] p update, [1] its barrier, [2] SpMV + <p,Ap>, [3] barrier + sum, [4] scalars + fused update,
 *                [5] barrier + sum;
 *   BiCGStab-M:  [0] SpMV#1 + <r0,q>, [1] barrier + sum, [2] scalars + s update, [3] barrier, [4] SpMV#2 + dots,
 *                [5] barrier + sum, [6] scalars + fused update, [7] barrier + sum;
 *   [15] iterations counted.  A barrier entry is what CTA 0 waits: the barrier itself plus the skew of the other
 * CTAs.  The other paths ignore it (msolve_profile_iteration times the kernels of the graph path).
 * d_ns = NULL switches it off (default).  Returns OK / EINVAL.  Table: profiles/r02_sweeps.md section 3. */
int msolve_set_phase_clock(msolve_matrix *A, uint64_t *d_ns);

/* ---------------------------------------------------------------------------------------------------------------
 * Row (site) partition: every slab owns a contiguous range of rows of A and the same range of r, p
 * and of every x_k, p_k.  Per iteration the halo of the gathered vector (p; BiCGStab-M also s) is exchanged before
 * each SpMV and the fused dot products are summed over the slabs; the fused multishift update (Alg. 1 l.28-29,
 * PAPER.md:129-131) needs no communication.  (The paper itself used one of its four GPUs.)
 *
 * msolve_slab_plan_*: HOST ONLY, no CUDA call.  The plan of slab `rank` of `nslabs`: rows [h_splits[rank],
 * h_splits[rank+1]) of an n x n matrix, given as the slab's own rows in CSR form (h_rowptr rebased to 0, GLOBAL
 * column indices).  It holds the off-slab columns the slab needs, grouped by owning slab (ascending) and sorted
 * within a slab -- halo entry j, at position nlocal + j of the slab's vectors -- and the slab's column indices
 * renumbered [own rows 0..nlocal-1 | halo nlocal..nlocal+nhalo-1].  What slab p must SEND to slab q is slab q's
 * list for peer p; ranks of a multi-process run exchange those lists once at set-up.
 * For BSR3 matrices the plan is built on block rows / block columns (indices count 3x3 blocks).
 * Errors: EINVAL (bad splits, column out of range, NULL), ENOMEM. */
typedef struct msolve_slab_plan msolve_slab_plan;
int msolve_slab_plan_create(msolve_slab_plan **plan, int64_t n, int nslabs, const int64_t *h_splits /* nslabs+1 */,
                            int rank, const int32_t *h_rowptr /* nlocal+1 */, const int32_t *h_colidx);
int64_t msolve_slab_plan_nlocal(const msolve_slab_plan *plan);
int64_t msolve_slab_plan_nhalo(const msolve_slab_plan *plan);
int msolve_slab_plan_npeers(const msolve_slab_plan *plan);
/* peer j (0 <= j < npeers): its rank, where its entries start in the halo, how many, and their GLOBAL column
 * indices (ascending; owned by the plan).  Any output pointer may be NULL. */
int msolve_slab_plan_peer(const msolve_slab_plan *plan, int j, int *peer_rank, int64_t *halo_offset, int64_t *count,
                          const int32_t **h_global_ids);
const int32_t *msolve_slab_plan_colidx(const msolve_slab_plan *plan); /* nnz renumbered columns (owned by the plan) */
void msolve_slab_plan_destroy(msolve_slab_plan *plan);

/* msolve_slabs_*: `nslabs` slabs of one matrix on the CURRENT device, in one process.  The matrix comes as HOST
 * arrays (the partitioner is host logic); the library keeps device copies of every slab's renumbered rows and one
 * ordinary handle per slab (same kernels as msolve_create_csr / msolve_create_bsr3 with the same `flags`).
 * h_splits: nslabs+1 row boundaries (block rows for BSR3), 16-byte aligned in the vectors, or NULL for an even
 * split.  The halo travels by a gather kernel that stores straight into the receiving slab's vector; the dot
 * products are summed over the slabs' per-CTA partials in fixed slab order; every slab repeats the scalar
 * recurrences on the same sums; the whole multi-slab iteration is one WHILE graph.  Arguments of the solvers as
 * msolve_cgm / msolve_bicgstabm with GLOBAL vectors (d_b: n, d_x: nshifts*n shift-major) and a workspace of
 * msolve_slabs_workspace_bytes().  Results agree with the unpartitioned solve to rounding (the dot products are
 * grouped by slab), and are bit-reproducible for a given number of slabs.  The slab set has no options: per-shift
 * stop rule, graph of kernels, no scalar history. */
typedef struct msolve_slabs msolve_slabs;
int msolve_slabs_create_csr(msolve_slabs **S, int64_t n, int64_t nnz, const int32_t *h_rowptr, const int32_t *h_colidx,
                            const void *h_val, int dtype, int nslabs, const int64_t *h_splits, int flags, void *stream);
int msolve_slabs_create_bsr3(msolve_slabs **S, int64_t nbrows, int64_t nblocks, const int32_t *h_browptr,
                             const int32_t *h_bcolidx, const void *h_blocks, int dtype, int nslabs,
                             const int64_t *h_splits, int flags, void *stream);
int msolve_slabs_count(const msolve_slabs *S);
int64_t msolve_slabs_halo_elements(const msolve_slabs *S, int slab); /* elements slab `slab` receives per exchange */
size_t msolve_slabs_workspace_bytes(const msolve_slabs *S, int nshifts, int algorithm);
int msolve_slabs_cgm(msolve_slabs *S, const void *d_b, const double *h_shifts, int nshifts, double tol, int max_iter,
                     void *d_x, void *d_workspace, size_t workspace_bytes, int *h_iterations, int *h_conv_iter,
                     double *h_relres, void *stream);
int msolve_slabs_bicgstabm(msolve_slabs *S, const void *d_b, const double *h_shifts, int nshifts, double tol,
                           int max_iter, void *d_x, void *d_workspace, size_t workspace_bytes, int *h_iterations,
                           int *h_conv_iter, double *h_relres, void *stream);
/* y = A x over the slabs (halo exchange + every slab's SpMV), h_dot = <x, A x>; workspace as for one shift of CG-M */
int msolve_slabs_spmv(msolve_slabs *S, const void *d_x, void *d_y, void *d_workspace, size_t workspace_bytes,
                      double *h_dot, void *stream);
int64_t msolve_slabs_last_launch_count(const msolve_slabs *S);
void msolve_slabs_destroy(msolve_slabs *S);

/* Free the handle and everything the library allocated for it (never the caller's arrays). */
void msolve_destroy(msolve_matrix *A);

/* Text of the last error on this thread ("" if none).  Never NULL. */
const char *msolve_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MSOLVE_H */
