"""Pins for the NEXT-3 (second half) oracle functions gram_cov and pca_transform
(PAPER.md:L95): numpy.cov on the dense matrix, an explicit loop on tiny inputs, symmetry / PSD,
the diagonal against the already pinned gene_moments, special cases."""
import numpy as np
import pytest

from oracle import oracle_np as O
from paper_2603_02402_b200 import synth


def _log_csr(n, G, seed, depth, **kw):
    indptr, indices, data, dense = synth.small_nb_csr(n, G, seed, depth, **kw)
    dl = np.log1p(data.astype(np.float64)).astype(np.float32)
    X = np.zeros((n, G)); X[np.repeat(np.arange(n), np.diff(indptr)), indices] = dl
    return indptr, indices, dl, X


@pytest.mark.parametrize("n,G,seed,depth", [(40, 30, 0, 2.0), (300, 90, 1, 0.7), (1000, 64, 2, 0.3)])
def test_gram_cov_against_numpy_cov(n, G, seed, depth):
    ip, ix, dl, X = _log_csr(n, G, seed, depth, empty_genes=(2,))
    r = O.gram_cov(ip, ix, dl, G)
    want = np.cov(X, rowvar=False)                       # centres explicitly, divides by n - 1
    np.testing.assert_allclose(r["cov"], want, rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(r["mean"], X.mean(axis=0), rtol=1e-13, atol=0)
    assert np.array_equal(r["gram"], r["gram"].T) or np.allclose(r["gram"], r["gram"].T, rtol=1e-15, atol=0)
    assert np.linalg.eigvalsh(r["cov"]).min() > -1e-10
    # the diagonal is the per-gene variance the moments oracle gives (ddof 1)
    _, var, s1, s2 = O.gene_moments(ip, ix, dl, G, 0, 1)
    np.testing.assert_allclose(np.diag(r["cov"]), var, rtol=1e-9, atol=1e-13)
    np.testing.assert_allclose(np.diag(r["gram"]), s2, rtol=1e-12)
    assert np.all(r["cov"][2] == 0) and np.all(r["cov"][:, 2] == 0)   # empty gene


def test_gram_explicit_loops_tiny():
    ip, ix, dl, X = _log_csr(12, 7, 5, 1.5)
    r = O.gram_cov(ip, ix, dl, 7)
    n = 12
    for a in range(7):
        for b in range(7):
            s = 0.0
            for i in range(n):
                s += X[i, a] * X[i, b]
            assert abs(r["gram"][a, b] - s) <= 1e-12 * max(1.0, abs(s))
            mu_a, mu_b = sum(X[:, a]) / n, sum(X[:, b]) / n
            c = sum((X[i, a] - mu_a) * (X[i, b] - mu_b) for i in range(n)) / (n - 1)
            assert abs(r["cov"][a, b] - c) <= 1e-11 * max(1.0, abs(c))


def test_gram_gene_permutation_and_constant_column():
    ip, ix, dl, X = _log_csr(60, 20, 7, 1.0)
    r = O.gram_cov(ip, ix, dl, 20)
    perm = np.random.default_rng(0).permutation(20)
    inv = np.argsort(perm)                               # new column of old gene g
    # relabel genes: sort each row's new indices to keep the CSR canonical
    ix2, d2 = ix.copy(), dl.copy()
    for i in range(60):
        s, e = ip[i], ip[i + 1]
        new = inv[ix[s:e]]
        o = np.argsort(new)
        ix2[s:e], d2[s:e] = new[o], dl[s:e][o]
    r2 = O.gram_cov(ip, ix2, d2, 20)
    np.testing.assert_allclose(r2["cov"], r["cov"][np.ix_(perm, perm)], rtol=1e-12, atol=1e-15)
    # a gene with the same value in every cell has zero covariance with everything
    n = 30
    ipc = np.arange(0, 2 * n + 1, 2, dtype=np.int64)
    ixc = np.tile(np.array([0, 3], dtype=np.int32), n)
    dc = np.empty(2 * n, dtype=np.float32); dc[0::2] = 1.25; dc[1::2] = np.arange(n, dtype=np.float32)
    rc = O.gram_cov(ipc, ixc, dc, 5)
    assert np.allclose(rc["cov"][0], 0, atol=1e-12) and np.isclose(rc["cov"][3, 3], np.var(np.arange(n), ddof=1))


@pytest.mark.parametrize("k", [1, 5])
def test_pca_transform(k):
    ip, ix, dl, X = _log_csr(80, 25, 3, 1.0)
    rng = np.random.default_rng(1)
    V = rng.standard_normal((25, k))
    mu = X.mean(axis=0)
    Z = O.pca_transform(ip, ix, dl, 25, V, mu)
    np.testing.assert_allclose(Z, (X - mu[None, :]) @ V, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(Z.sum(axis=0), 0, atol=1e-9)
    Zi = O.pca_transform(ip, ix, dl, 25, np.eye(25), mu)
    np.testing.assert_allclose(Zi, X - mu[None, :], rtol=1e-13, atol=1e-15)
    # eigenvectors of the oracle covariance: projected coordinates have the eigenvalues as variances
    C = O.gram_cov(ip, ix, dl, 25)["cov"]
    w, U = np.linalg.eigh(C)
    Zp = O.pca_transform(ip, ix, dl, 25, U[:, -3:], mu)
    np.testing.assert_allclose(Zp.var(axis=0, ddof=1), w[-3:], rtol=1e-9)
