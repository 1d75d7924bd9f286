"""Seeded synthetic workloads for the multishift solvers (input generators ONLY).

This module builds the inputs of BASELINE.json's five configs (and scaled-down /
pin variants of them) from a seed: sparse matrices A in CSR and 3x3-block BSR form,
right-hand sides b and shift arrays sigma.  It contains none of the method's
arithmetic (no SpMV, no dot, no recurrence, no solver) and is the only code that
serves both the CPU oracle (``oracle/``) and the CUDA path: both receive the very
same host arrays.  The recipe is the one written down in DESIGN.md ("Input recipe")
after SURVEY.md section 8(d).

Conventions
-----------
* Lattice sites: extents (L0, ..., L_{d-1}), dimension 0 fastest,
  site s = x0 + L0*(x1 + L1*(...)); periodic in every direction.
* SU(3) operators: row = 3*s + colour.  Block (s, s+mu) = -c_f * U_mu(s),
  block (s, s-mu) = -c_b * U_mu(s-mu)^dagger, diagonal block D * I_3 (stored as a
  full 3x3 block, so the CSR row expansion has 27 stored entries per row, 2 of
  them explicit zeros -- BASELINE.json's "27 nnz/row").
* Block columns are sorted ascending inside every block row; CSR is the
  row expansion of exactly the same blocks.
* All generation is complex128; complex64 runs cast the finished arrays.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Optional, Sequence, Tuple

import numpy as np

DEFAULT_SEED = 11022143  # arXiv number of the paper; fixed for the repo


# --------------------------------------------------------------------------- rng
def _substream(seed: int, name: str) -> np.random.Generator:
    """Independent generator for one named sub-stream (links, b, pattern, values)."""
    tag = int.from_bytes(name.encode()[:8].ljust(8, b"\0"), "little")
    return np.random.Generator(np.random.Philox(np.random.SeedSequence([seed, tag])))


def complex_gaussian(rng: np.random.Generator, shape) -> np.ndarray:
    """Standard complex normal: E|z|^2 = 1."""
    z = rng.standard_normal(size=tuple(np.atleast_1d(shape)) + (2,))
    return (z[..., 0] + 1j * z[..., 1]) * np.sqrt(0.5)


def unit_rhs(seed: int, n: int) -> np.ndarray:
    """b: complex Gaussian normalised to ||b|| = 1 (every config)."""
    b = complex_gaussian(_substream(seed, "b"), n)
    return b / np.sqrt(np.sum(b.real ** 2 + b.imag ** 2))


def real_unit_rhs(seed: int, n: int) -> np.ndarray:
    """b: real Gaussian, ||b|| = 1 (the paper's own runs are real-valued)."""
    b = _substream(seed, "b").standard_normal(n)
    return b / np.sqrt(np.sum(b * b))


def log_shifts(lo: float, hi: float, count: int) -> np.ndarray:
    """`count` points log-spaced from lo to hi, endpoints included."""
    return np.logspace(np.log10(lo), np.log10(hi), count).astype(np.float64)


# ----------------------------------------------------------------------- lattice
def neighbour_tables(extents: Sequence[int]) -> Tuple[np.ndarray, np.ndarray]:
    """fwd[mu, s] = index of s+mu, bwd[mu, s] = index of s-mu (periodic)."""
    ext = tuple(int(e) for e in extents)
    if min(ext) < 3:
        raise ValueError("extents must be >= 3 (forward and backward neighbours must differ)")
    d = len(ext)
    vol = int(np.prod(ext))
    idx = np.arange(vol, dtype=np.int64).reshape(ext[::-1])  # last axis = dimension 0
    fwd = np.empty((d, vol), dtype=np.int64)
    bwd = np.empty((d, vol), dtype=np.int64)
    for mu in range(d):
        ax = d - 1 - mu
        fwd[mu] = np.roll(idx, -1, axis=ax).ravel()
        bwd[mu] = np.roll(idx, +1, axis=ax).ravel()
    return fwd, bwd


def haar_su3(rng: np.random.Generator, count: int) -> np.ndarray:
    """`count` Haar-random SU(3) matrices, shape (count, 3, 3).

    3x3 complex Ginibre -> QR with positive diagonal of R (written as Gram-Schmidt
    on the columns, which is that QR) -> divide by det^(1/3) (principal root).
    """
    z = complex_gaussian(rng, (count, 3, 3))
    q = np.empty_like(z)
    c0 = z[:, :, 0]
    q0 = c0 / np.linalg.norm(c0, axis=1, keepdims=True)
    c1 = z[:, :, 1]
    c1 = c1 - q0 * np.sum(q0.conj() * c1, axis=1, keepdims=True)
    q1 = c1 / np.linalg.norm(c1, axis=1, keepdims=True)
    c2 = z[:, :, 2]
    c2 = c2 - q0 * np.sum(q0.conj() * c2, axis=1, keepdims=True)
    c2 = c2 - q1 * np.sum(q1.conj() * c2, axis=1, keepdims=True)
    q2 = c2 / np.linalg.norm(c2, axis=1, keepdims=True)
    q[:, :, 0], q[:, :, 1], q[:, :, 2] = q0, q1, q2
    det = (q[:, 0, 0] * (q[:, 1, 1] * q[:, 2, 2] - q[:, 1, 2] * q[:, 2, 1])
           - q[:, 0, 1] * (q[:, 1, 0] * q[:, 2, 2] - q[:, 1, 2] * q[:, 2, 0])
           + q[:, 0, 2] * (q[:, 1, 0] * q[:, 2, 1] - q[:, 1, 1] * q[:, 2, 0]))
    phase = np.exp(-1j * np.angle(det) / 3.0)
    return q * phase[:, None, None]


def su3_links(seed: int, extents: Sequence[int], kind: str = "haar") -> np.ndarray:
    """links[mu, s] = U_mu(s), shape (d, V, 3, 3).

    kind="haar": independent Haar SU(3) per link (the BASELINE configs).
    kind="pure_gauge": U_mu(s) = g(s) g(s+mu)^dagger with Haar g(s) -- a gauge
    transform of the free field, used only by the FFT closed-form pin.
    """
    fwd, _ = neighbour_tables(extents)
    d, vol = fwd.shape
    rng = _substream(seed, "links")
    if kind == "haar":
        return haar_su3(rng, d * vol).reshape(d, vol, 3, 3)
    if kind == "pure_gauge":
        g = haar_su3(rng, vol)
        links = np.empty((d, vol, 3, 3), dtype=np.complex128)
        for mu in range(d):
            links[mu] = g @ np.conj(np.swapaxes(g[fwd[mu]], 1, 2))
        return links
    raise ValueError(kind)


def gauged_operator_bsr3(extents: Sequence[int], links: np.ndarray, diag: float,
                         c_f: float, c_b: float):
    """A = diag*I - sum_mu ( c_f U_mu(s) delta_{s+mu,t} + c_b U_mu(s-mu)^dagger delta_{s-mu,t} ).

    Returns (browptr int32 [V+1], bcolidx int32 [9V... (2d+1)V], blocks complex128 [nb,3,3]),
    block columns ascending inside each block row.
    """
    fwd, bwd = neighbour_tables(extents)
    d, vol = fwd.shape
    per = 2 * d + 1
    cols = np.empty((vol, per), dtype=np.int64)
    blocks = np.empty((vol, per, 3, 3), dtype=np.complex128)
    cols[:, 0] = np.arange(vol)
    blocks[:, 0] = diag * np.eye(3)
    for mu in range(d):
        cols[:, 1 + 2 * mu] = fwd[mu]
        blocks[:, 1 + 2 * mu] = -c_f * links[mu]
        cols[:, 2 + 2 * mu] = bwd[mu]
        blocks[:, 2 + 2 * mu] = -c_b * np.conj(np.swapaxes(links[mu][bwd[mu]], 1, 2))
    order = np.argsort(cols, axis=1, kind="stable")
    cols = np.take_along_axis(cols, order, axis=1)
    blocks = np.take_along_axis(blocks, order[:, :, None, None], axis=1)
    browptr = (np.arange(vol + 1, dtype=np.int64) * per).astype(np.int32)
    return browptr, cols.reshape(-1).astype(np.int32), blocks.reshape(-1, 3, 3)


def bsr3_to_csr(browptr: np.ndarray, bcolidx: np.ndarray, blocks: np.ndarray):
    """Row expansion of a 3x3-block matrix (keeps explicit zeros, keeps ordering)."""
    nbrows = browptr.size - 1
    cnt = np.diff(browptr.astype(np.int64))
    per = int(cnt[0]) if nbrows else 0
    if nbrows and np.all(cnt == per):  # regular (lattice) fast path
        bl = blocks.reshape(nbrows, per, 3, 3).transpose(0, 2, 1, 3)  # (site, r, slot, c)
        val = np.ascontiguousarray(bl).reshape(-1)
        bc = bcolidx.reshape(nbrows, per).astype(np.int64)
        col = (3 * bc[:, None, :, None] + np.arange(3)[None, None, None, :])
        col = np.broadcast_to(col, (nbrows, 3, per, 3)).reshape(-1)
        rowptr = np.arange(3 * nbrows + 1, dtype=np.int64) * (3 * per)
        return rowptr.astype(np.int32), col.astype(np.int32), val
    rowptr = np.zeros(3 * nbrows + 1, dtype=np.int64)
    rowptr[1:] = np.cumsum(np.repeat(3 * cnt, 3))
    col = np.empty(int(rowptr[-1]), dtype=np.int32)
    val = np.empty(int(rowptr[-1]), dtype=np.complex128)
    for br in range(nbrows):  # general, small inputs only
        lo, hi = int(browptr[br]), int(browptr[br + 1])
        for r in range(3):
            o = int(rowptr[3 * br + r])
            for t, k in enumerate(range(lo, hi)):
                col[o + 3 * t:o + 3 * t + 3] = 3 * int(bcolidx[k]) + np.arange(3)
                val[o + 3 * t:o + 3 * t + 3] = blocks[k, r, :]
    return rowptr.astype(np.int32), col, val


def u1_operator_csr(seed: int, extents: Sequence[int], diag: float):
    """Config 1: A = diag*I - sum_mu ( U_mu(s) delta_{s+mu,t} + h.c. ), U = exp(i theta)."""
    fwd, bwd = neighbour_tables(extents)
    d, vol = fwd.shape
    theta = _substream(seed, "links").uniform(0.0, 2.0 * np.pi, size=(d, vol))
    u = np.exp(1j * theta)
    per = 2 * d + 1
    cols = np.empty((vol, per), dtype=np.int64)
    vals = np.empty((vol, per), dtype=np.complex128)
    cols[:, 0] = np.arange(vol)
    vals[:, 0] = diag
    for mu in range(d):
        cols[:, 1 + 2 * mu] = fwd[mu]
        vals[:, 1 + 2 * mu] = -u[mu]
        cols[:, 2 + 2 * mu] = bwd[mu]
        vals[:, 2 + 2 * mu] = -np.conj(u[mu][bwd[mu]])
    order = np.argsort(cols, axis=1, kind="stable")
    cols = np.take_along_axis(cols, order, axis=1)
    vals = np.take_along_axis(vals, order, axis=1)
    rowptr = (np.arange(vol + 1, dtype=np.int64) * per).astype(np.int32)
    return rowptr, cols.reshape(-1).astype(np.int32), vals.reshape(-1)


def poisson5pt_csr(nx: int, ny: int, dtype=np.complex128, drift: float = 0.0):
    """The paper's own test matrix: 2-D 5-point Laplacian, Dirichlet.

    drift != 0 adds a centred first-derivative term in x (east -1+drift, west -1-drift): a real
    NON-symmetric convection-diffusion matrix, the real-valued input of the BiCGStab-M tests.
    """
    idx = np.arange(nx * ny, dtype=np.int64).reshape(ny, nx)
    rows, cols, vals = [idx.ravel()], [idx.ravel()], [np.full(nx * ny, 4.0)]
    for (sl_a, sl_b), d in ((((slice(None), slice(0, nx - 1)), (slice(None), slice(1, nx))), drift),
                            (((slice(0, ny - 1), slice(None)), (slice(1, ny), slice(None))), 0.0)):
        a, b = idx[sl_a].ravel(), idx[sl_b].ravel()
        rows += [a, b]
        cols += [b, a]
        vals += [np.full(a.size, -1.0 + d), np.full(a.size, -1.0 - d)]
    return coo_to_csr(nx * ny, np.concatenate(rows), np.concatenate(cols),
                      np.concatenate(vals).astype(dtype))


def coo_to_csr(n: int, rows: np.ndarray, cols: np.ndarray, vals: np.ndarray):
    """Sort (row, col) ascending and build rowptr.  No duplicate handling."""
    key = rows.astype(np.int64) * n + cols.astype(np.int64)
    order = np.argsort(key, kind="stable")
    rows, cols, vals = rows[order], cols[order], vals[order]
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(np.bincount(rows, minlength=n), out=rowptr[1:])
    if rowptr[-1] >= 2 ** 31:
        raise ValueError("nnz does not fit int32 indices")
    return rowptr.astype(np.int32), cols.astype(np.int32), vals


# ------------------------------------------------------------------ unstructured
def _powerlaw_gamma(lo: int, hi: int, mean: float) -> float:
    ell = np.arange(lo, hi + 1, dtype=np.float64)

    def m(g):
        w = ell ** (-g)
        return float(np.sum(ell * w) / np.sum(w))

    a, b = 0.0, 6.0
    for _ in range(200):
        mid = 0.5 * (a + b)
        if m(mid) > mean:
            a = mid
        else:
            b = mid
    return 0.5 * (a + b)


def powerlaw_hpd_csr(seed: int, n: int, lo: int = 5, hi: int = 200, mean: float = 32.0):
    """Config 5: Hermitian positive-definite CSR with power-law row lengths.

    Row length l_i (diagonal included) ~ P(l) ∝ l^-gamma on [lo, hi], gamma solved so the
    mean is `mean`; symmetric pattern by the configuration model (stubs shuffled and
    paired, self-pairs and duplicates dropped, short rows topped up); off-diagonals
    complex Gaussian mirrored as conjugates; diagonal = sum_j |a_ij| + 0.01.
    """
    gamma = _powerlaw_gamma(lo, hi, mean)
    ell = np.arange(lo, hi + 1)
    w = ell.astype(np.float64) ** (-gamma)
    cdf = np.cumsum(w) / np.sum(w)
    rng = _substream(seed, "pattern")
    length = ell[np.searchsorted(cdf, rng.random(n), side="left").clip(0, ell.size - 1)]
    stubs = np.repeat(np.arange(n, dtype=np.int64), length - 1)
    stubs = stubs[rng.permutation(stubs.size)]
    stubs = stubs[: stubs.size - (stubs.size & 1)]
    a, b = stubs[0::2], stubs[1::2]

    def canon(a, b):
        keep = a != b
        a, b = a[keep], b[keep]
        lo_, hi_ = np.minimum(a, b), np.maximum(a, b)
        return np.unique(lo_ * n + hi_)

    key = canon(a, b)
    for _ in range(4):  # top up rows that fell below lo-1 off-diagonals
        deg = np.bincount(key // n, minlength=n) + np.bincount(key % n, minlength=n)
        short = np.flatnonzero(deg < lo - 1)
        if short.size == 0:
            break
        need = np.repeat(short, (lo - 1) - deg[short])
        partner = rng.integers(0, n, size=need.size)
        key = np.unique(np.concatenate([key, canon(need, partner)]))
    ei, ej = key // n, key % n
    aij = complex_gaussian(_substream(seed, "values"), ei.size)
    absum = (np.bincount(ei, weights=np.abs(aij), minlength=n)
             + np.bincount(ej, weights=np.abs(aij), minlength=n))
    rows = np.concatenate([ei, ej, np.arange(n, dtype=np.int64)])
    cols = np.concatenate([ej, ei, np.arange(n, dtype=np.int64)])
    vals = np.concatenate([aij, np.conj(aij), (absum + 0.01).astype(np.complex128)])
    return coo_to_csr(n, rows, cols, vals)


# ---------------------------------------------------------------------- workload
@dataclass
class Workload:
    """One solver problem: everything `msolve_cgm` / `msolve_bicgstabm` is given."""
    name: str
    algorithm: str                 # "cgm" | "bicgstabm"
    n: int
    shifts: np.ndarray             # float64 [S]
    tol: float
    max_iter: int
    b: np.ndarray                  # complex128 [n], unit norm
    rowptr: np.ndarray             # int32 [n+1]
    colidx: np.ndarray             # int32 [nnz]
    val: np.ndarray                # complex128 [nnz]
    browptr: Optional[np.ndarray] = None   # int32 [n/3+1]
    bcolidx: Optional[np.ndarray] = None   # int32 [nb]
    blocks: Optional[np.ndarray] = None    # complex128 [nb,3,3]
    links: Optional[np.ndarray] = None     # complex128 [d,V,3,3], links[mu,s] = U_mu(s) (lattice workloads)
    meta: Dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.colidx.size)

    @property
    def has_bsr3(self) -> bool:
        return self.blocks is not None


def su3_workload(name: str, algorithm: str, extents: Sequence[int], diag: float, c_f: float,
                 c_b: float, shifts: np.ndarray, tol: float, seed: int = DEFAULT_SEED,
                 max_iter: int = 2000, links: str = "haar", want_csr: bool = True) -> Workload:
    lk = su3_links(seed, extents, links)
    browptr, bcolidx, blocks = gauged_operator_bsr3(extents, lk, diag, c_f, c_b)
    n = 3 * (browptr.size - 1)
    if want_csr:
        rowptr, colidx, val = bsr3_to_csr(browptr, bcolidx, blocks)
    else:
        rowptr = colidx = val = np.zeros(0)
    return Workload(name, algorithm, n, np.asarray(shifts, dtype=np.float64), tol, max_iter,
                    unit_rhs(seed, n), rowptr, colidx, val, browptr, bcolidx, blocks, lk,
                    {"extents": tuple(extents), "diag": diag, "c_f": c_f, "c_b": c_b,
                     "links": links, "seed": seed})


def config1(seed: int = DEFAULT_SEED, extents=(8, 8)) -> Workload:
    """CG-M, 2-D U(1) lattice, m=0.1, shifts {0,.01,.1,1}, tol 1e-10."""
    m = 0.1
    rowptr, colidx, val = u1_operator_csr(seed, extents, m * m + 2 * len(extents))
    n = rowptr.size - 1
    return Workload("config1_u1_%s" % "x".join(map(str, extents)), "cgm", n,
                    np.array([0.0, 0.01, 0.1, 1.0]), 1e-10, 2000, unit_rhs(seed, n),
                    rowptr, colidx, val, meta={"extents": tuple(extents), "seed": seed})


def config2(seed: int = DEFAULT_SEED, extents=(8, 8, 8, 8), links="haar") -> Workload:
    """CG-M, 4-D SU(3) gauged Laplacian, m=0.05, 12 shifts 1e-4..1, tol 1e-10."""
    m = 0.05
    return su3_workload("config2_su3_%s" % "x".join(map(str, extents)), "cgm", extents,
                        m * m + 2 * len(extents), 1.0, 1.0, log_shifts(1e-4, 1.0, 12), 1e-10,
                        seed, links=links)


def config3(seed: int = DEFAULT_SEED, extents=(16, 16, 16, 16), links="haar") -> Workload:
    """BiCGStab-M, non-Hermitian 4-D SU(3) operator, m=0.2, 8 shifts, tol 1e-9."""
    m = 0.2
    shifts = np.array([0.0, 0.02, 0.05, 0.1, 0.2, 0.5, 1.0, 2.0])
    return su3_workload("config3_su3nh_%s" % "x".join(map(str, extents)), "bicgstabm", extents,
                        len(extents) + m, 0.6, 0.4, shifts, 1e-9, seed, links=links)


def config4(seed: int = DEFAULT_SEED, extents=(32, 32, 32, 64), tol: float = 1e-10,
            want_csr: bool = True, links="haar") -> Workload:
    """CG-M, 32^3x64 SU(3) gauged Laplacian, m=0.02, 16 shifts 1e-5..1."""
    m = 0.02
    return su3_workload("config4_su3_%s" % "x".join(map(str, extents)), "cgm", extents,
                        m * m + 2 * len(extents), 1.0, 1.0, log_shifts(1e-5, 1.0, 16), tol,
                        seed, want_csr=want_csr, links=links)


def config5(seed: int = DEFAULT_SEED, n: int = 1 << 22, tol: float = 1e-10) -> Workload:
    """CG-M, unstructured Hermitian PD CSR, power-law rows, 32 shifts 1e-3..10."""
    rowptr, colidx, val = powerlaw_hpd_csr(seed, n)
    return Workload("config5_powerlaw_%d" % n, "cgm", n, log_shifts(1e-3, 10.0, 32), tol, 5000,
                    unit_rhs(seed, n), rowptr, colidx, val, meta={"seed": seed})


def poisson_workload(nx: int, ny: int, nshifts: int = 15, tol: float = 1e-5,
                     seed: int = DEFAULT_SEED, real: bool = False, drift: float = 0.0) -> Workload:
    """The paper's Table-1 workload shape: 2-D Poisson, 15 shifts (the paper does
    not state their values: log-spaced 1e-3..1 here).  real=True: float64 matrix and right-hand
    side, as the paper ran it; otherwise the same numbers stored as complex.  drift != 0: the
    non-symmetric variant for BiCGStab-M."""
    rowptr, colidx, val = poisson5pt_csr(nx, ny, np.float64 if real else np.complex128, drift)
    n = nx * ny
    b = real_unit_rhs(seed, n) if real else unit_rhs(seed, n)
    return Workload("poisson5pt_%dx%d%s" % (nx, ny, "_drift" if drift else ""),
                    "bicgstabm" if drift else "cgm", n, log_shifts(1e-3, 1.0, nshifts), tol,
                    20000, b, rowptr, colidx, val, meta={"nx": nx, "ny": ny, "drift": drift})
