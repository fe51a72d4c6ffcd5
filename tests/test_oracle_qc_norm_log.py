"""Pins for the oracle's QC / normalize_total / log1p (Q1..Q4, N1, L1).

Every expected value here comes from something OTHER than the oracle: explicit
loops over the dense matrix, scipy.sparse / numpy library reductions, closed
forms, and the invariants BASELINE.json's north_star names.
"""
import numpy as np
import pytest
import scipy.sparse as sp

from oracle import oracle_np as O
from paper_2603_02402_b200 import synth

CASES = [  # n, G, seed, depth, empty_rows, empty_genes
    (1, 1, 0, 3.0, (), ()),
    (7, 5, 1, 2.0, (3,), (2,)),
    (40, 33, 2, 1.0, (0, 39), (0, 32)),
    (64, 200, 3, 0.5, (), (5, 6, 7)),
    (130, 97, 4, 1.5, (17,), ()),
]


def _flags(G, seed):
    rng = np.random.default_rng(100 + seed)
    return (rng.random(G) < 0.3).astype(np.uint8)


@pytest.mark.parametrize("n,G,seed,depth,er,eg", CASES)
def test_qc_dense_bruteforce(n, G, seed, depth, er, eg):
    indptr, indices, data, X = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    flags = _flags(G, seed)
    q = O.qc_metrics(indptr, indices, data, G, flags)
    # explicit loops over the dense matrix
    for i in range(n):
        T = 0; N = 0; M = 0
        for j in range(G):
            x = int(X[i, j])
            T += x
            N += 1 if X[i, j] != 0 else 0
            if flags[j]:
                M += x
        assert q["cell_total_i64"][i] == T
        assert q["cell_n_genes"][i] == N
        assert q["cell_flag_total_i64"][i] == M
        assert q["cell_total_f32"][i] == np.float32(T)
        if T == 0:
            assert np.isnan(q["cell_flag_pct"][i])
        else:
            assert q["cell_flag_pct"][i] == np.float32(100.0 * M / T)
    for j in range(G):
        assert q["gene_n_cells"][j] == int(np.count_nonzero(X[:, j]))
        assert q["gene_total_i64"][j] == int(X[:, j].sum())
    assert q["cell_total_i64"].dtype == np.int64 and q["gene_n_cells"].dtype == np.int32


@pytest.mark.parametrize("n,G,seed,depth,er,eg", CASES)
def test_qc_scipy_and_invariants(n, G, seed, depth, er, eg):
    indptr, indices, data, X = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    q = O.qc_metrics(indptr, indices, data, G, None)
    A = sp.csr_matrix((data.astype(np.float64), indices, indptr), shape=(n, G))
    assert np.array_equal(q["cell_total_i64"], np.asarray(A.sum(axis=1)).ravel().astype(np.int64))
    assert np.array_equal(q["gene_total_i64"], np.asarray(A.sum(axis=0)).ravel().astype(np.int64))
    assert np.array_equal(q["gene_n_cells"], np.bincount(indices, minlength=G))
    assert np.array_equal(q["cell_n_genes"], np.diff(indptr))
    nnz = indices.shape[0]
    # north_star invariants: per-gene nnz counts add up to total nnz, both total sums agree
    assert q["cell_n_genes"].sum() == nnz == q["gene_n_cells"].sum()
    assert q["cell_total_i64"].sum() == q["gene_total_i64"].sum()
    assert np.all(q["cell_flag_total_i64"] == 0)      # no flags -> 0


def test_qc_flag_special_cases_and_explicit_zero():
    indptr, indices, data, X = synth.small_nb_csr(20, 15, 9, 2.0)
    allf = np.ones(15, np.uint8)
    q = O.qc_metrics(indptr, indices, data, 15, allf)
    ok = q["cell_total_i64"] > 0
    assert np.all(q["cell_flag_pct"][ok] == np.float32(100.0))
    q0 = O.qc_metrics(indptr, indices, data, 15, np.zeros(15, np.uint8))
    assert np.all(q0["cell_flag_pct"][ok] == 0.0)
    # an explicitly stored zero is not "detected" (reading R2)
    d2 = data.copy(); d2[0] = 0.0
    q2 = O.qc_metrics(indptr, indices, d2, 15, None)
    assert q2["cell_n_genes"][0] == q["cell_n_genes"][0] - 1
    assert q2["gene_n_cells"][indices[0]] == q["gene_n_cells"][indices[0]] - 1


@pytest.mark.parametrize("n,G,seed,depth,er,eg", CASES)
@pytest.mark.parametrize("s", [1e4, 1e6, 37.5])
def test_normalize_total(n, G, seed, depth, er, eg, s):
    indptr, indices, data, X = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    xn, scale = O.normalize_total(indptr, data, s, None)
    assert xn.dtype == np.float32
    T = X.sum(axis=1)
    # dense brute force, paper's formula (x / sum) * s
    for i in range(n):
        lo, hi = indptr[i], indptr[i + 1]
        if T[i] == 0:
            assert hi == lo
            continue
        want = (X[i, indices[lo:hi]] / T[i]) * s
        np.testing.assert_allclose(xn[lo:hi], want, rtol=3e-7, atol=0)
        # invariant: row sums equal target_sum
        rs = xn[lo:hi].astype(np.float64).sum()
        assert abs(rs - s) <= s * (hi - lo) * 2.0 ** -24
    # supplying the exact totals gives the identical result
    q = O.qc_metrics(indptr, indices, data, G, None)
    xn2, _ = O.normalize_total(indptr, data, s, q["cell_total_i64"])
    assert np.array_equal(xn, xn2)


def test_normalize_identity_when_s_equals_total():
    # every row has total exactly 64 -> s = 64 leaves the data bit-identical
    indptr = np.array([0, 2, 5, 6], dtype=np.int64)
    indices = np.array([0, 3, 1, 2, 4, 0], dtype=np.int32)
    data = np.array([60, 4, 1, 3, 60, 64], dtype=np.float32)
    xn, scale = O.normalize_total(indptr, data, 64.0, None)
    assert np.array_equal(xn, data) and np.all(scale == 1.0)
    # empty cell: untouched, scale 1 (reading R3)
    indptr2 = np.array([0, 0, 2], dtype=np.int64)
    xn2, sc2 = O.normalize_total(indptr2, np.array([1, 3], np.float32), 100.0, None)
    assert sc2[0] == 1.0 and np.array_equal(xn2, np.array([25, 75], np.float32))


@pytest.mark.parametrize("n,G,seed,depth,er,eg", CASES)
def test_log1p(n, G, seed, depth, er, eg):
    indptr, indices, data, X = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    xn, _ = O.normalize_total(indptr, data, 1e4, None)
    xl = O.log1p(xn)
    assert xl.dtype == np.float32 and xl.shape == xn.shape
    # library pin: numpy.log1p on the dense normalised matrix
    D = np.zeros((n, G))
    rows = np.repeat(np.arange(n), np.diff(indptr))
    D[rows, indices] = xn
    L = np.log1p(D)
    np.testing.assert_allclose(xl, L[rows, indices], rtol=1e-7)
    # log1p(0) = 0 keeps the sparsity pattern: x'' = 0 <=> x' = 0
    assert np.array_equal(L == 0, D == 0)
    assert np.all((xl == 0) == (xn == 0))
    # round trip
    np.testing.assert_allclose(np.expm1(xl.astype(np.float64)), xn, rtol=2e-6)
    # hand values: log1p(e-1) = 1 ; log1p(0) = 0
    assert O.log1p(np.array([np.e - 1, 0.0], np.float32))[0] == np.float32(1.0)
    assert O.log1p(np.array([0.0], np.float32))[0] == 0.0
