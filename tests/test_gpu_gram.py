"""GPU parity of rsc_gram_cov (second half) against
oracle_np.gram_cov: mean at 1e-12, Gram matrix entry-wise at 1e-5 relative (the paper's own
allclose bar, L155; DESIGN.md section 6 gives the error budget of the fp16-pair tensor-core
contraction), covariance within the same absolute error divided by n - 1."""
import numpy as np
import pytest
import torch

from oracle import oracle_np as O
from paper_2603_02402_b200 import Csr, binding as B, synth

pytestmark = pytest.mark.gpu

GRAM_RTOL = 1e-5


def _log_csr(n, G, seed, depth, sort=True):
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth)
    dl = np.log1p(data.astype(np.float64)).astype(np.float32)
    if not sort:                                         # reverse every row: unsorted columns
        for i in range(n):
            s, e = indptr[i], indptr[i + 1]
            indices[s:e] = indices[s:e][::-1].copy()
            dl[s:e] = dl[s:e][::-1].copy()
    return indptr, indices, dl


def _check(ip, ix, dl, G, sorted_rows=True):
    X = Csr(torch.from_numpy(ip).cuda(), torch.from_numpy(ix).cuda(), torch.from_numpy(dl).cuda(), G,
            sorted_indices=sorted_rows)
    out = B.rsc_gram_cov(X)
    torch.cuda.synchronize()
    ref = O.gram_cov(ip, ix, dl, G)
    n = len(ip) - 1
    mean, S, Cv = out["mean"].cpu().numpy(), out["gram"].cpu().numpy(), out["cov"].cpu().numpy()
    np.testing.assert_allclose(mean, ref["mean"], rtol=1e-12, atol=0)
    assert np.array_equal(S, S.T) and np.array_equal(Cv, Cv.T)          # mirrored, bit for bit
    err = np.abs(S - ref["gram"])
    assert np.all(err <= GRAM_RTOL * np.abs(ref["gram"])), (err.max(), (err / np.maximum(np.abs(ref["gram"]), 1e-300)).max())
    assert np.all((ref["gram"] == 0) <= (S == 0))                       # structural zeros stay exact zeros
    cerr = np.abs(Cv - ref["cov"])
    bound = GRAM_RTOL * np.abs(ref["gram"]) / (n - 1) + 1e-12 * np.abs(ref["cov"]) + 1e-300
    assert np.all(cerr <= bound + 4e-16 * n * np.abs(np.outer(ref["mean"], ref["mean"])) / (n - 1))
    return out


@pytest.mark.parametrize("n,G,seed,depth", [(300, 100, 0, 1.0), (1000, 300, 1, 0.6), (4097, 700, 2, 0.4),
                                             (2500, 64, 3, 2.0), (33, 129, 4, 1.0)])
def test_gram_cov_small(n, G, seed, depth):
    ip, ix, dl = _log_csr(n, G, seed, depth)
    _check(ip, ix, dl, G)


def test_gram_cov_unsorted_rows_and_reproducible():
    ip, ix, dl = _log_csr(700, 260, 5, 0.8, sort=False)
    a = _check(ip, ix, dl, 260, sorted_rows=False)
    b = _check(ip, ix, dl, 260, sorted_rows=False)
    assert torch.equal(a["gram"], b["gram"]) and torch.equal(a["cov"], b["cov"])   # no atomics: same bits


def test_gram_cov_hvg_subset_of_cfg1():
    """raw counts -> chain -> HVG subset -> Gram / covariance, the workflow order of L47."""
    cfg = synth.scaled(synth.CONFIGS[1], 3000)
    indptr, indices, data = synth.make_csr(cfg, "cuda")
    flags = synth.gene_flags(cfg, "cuda")
    X = Csr(indptr, indices, data, cfg.n_genes)
    out = B.rsc_preprocess(X, flags, cfg.target_sum, 1500, cfg.n_bins)
    Y, g2 = B.rsc_subset_csr(X, None, out["hvg_mask"])
    torch.cuda.synchronize()
    ip, ix, dl = Y.indptr.cpu().numpy(), Y.indices.cpu().numpy(), Y.data.cpu().numpy()
    _check(ip, ix, dl, g2)


@pytest.mark.parametrize("n,G,k,seed,center", [(300, 100, 5, 0, True), (1000, 300, 50, 1, True), (777, 129, 33, 2, False),
                                               (2000, 500, 128, 3, True), (64, 40, 1, 4, True),
                                               # large loading tables (0.8 - 3 MB: served from L2), a short matrix
                                               (1500, 4000, 50, 5, True), (500, 2300, 128, 6, True),
                                               (200, 6000, 128, 7, False), (33, 4000, 50, 8, False)])
def test_pca_transform(n, G, k, seed, center):
    """rsc_pca_transform against oracle_np.pca_transform (PAPER.md:L95 Z = XV - 1 mu^T V).  Bound: V
    travels as float32 (6e-8 per term) and the result is rounded to float32."""
    ip, ix, dl = _log_csr(n, G, seed, 1.0)
    rng = np.random.default_rng(seed)
    V = np.linalg.qr(rng.standard_normal((G, k)))[0] if k <= G else rng.standard_normal((G, k))
    V = np.ascontiguousarray(V)
    X = Csr(torch.from_numpy(ip).cuda(), torch.from_numpy(ix).cuda(), torch.from_numpy(dl).cuda(), G)
    dense = np.zeros((n, G)); dense[np.repeat(np.arange(n), np.diff(ip)), ix] = dl
    mu = dense.mean(axis=0)
    Z = B.rsc_pca_transform(X, torch.from_numpy(V).cuda(), torch.from_numpy(mu).cuda() if center else None)
    torch.cuda.synchronize()
    ref = O.pca_transform(ip, ix, dl, G, V, mu if center else np.zeros(G))
    mass = np.abs(dense) @ np.abs(V) + (np.abs(mu) @ np.abs(V))[None, :] * (1 if center else 0)
    err = np.abs(Z.cpu().numpy() - ref)
    assert np.all(err <= 1e-7 * mass + 1.2e-7 * np.abs(ref) + 1e-30), err.max()


def test_gram_eigh_transform_workflow():
    """Gram -> covariance -> eigenvectors (torch.linalg.eigh: the library step the paper also uses)
    -> projection; the projected coordinates have the top eigenvalues as variances."""
    ip, ix, dl = _log_csr(3000, 200, 7, 0.8)
    X = Csr(torch.from_numpy(ip).cuda(), torch.from_numpy(ix).cuda(), torch.from_numpy(dl).cuda(), 200)
    g = B.rsc_gram_cov(X)
    w, U = torch.linalg.eigh(g["cov"])
    V = U[:, -10:].contiguous()
    Z = B.rsc_pca_transform(X, V, g["mean"]).double()
    np.testing.assert_allclose(Z.var(dim=0, unbiased=True).cpu().numpy(), w[-10:].cpu().numpy(), rtol=2e-5)
    assert float(Z.mean(dim=0).abs().max()) < 1e-5


def test_gram_cov_many_slabs_and_wide():
    """More cells than one pack / MMA slab (262 144): partial tiles accumulate across slabs; and
    more genes than 16 column tiles.  Random sparse log-like values drawn directly (no NB)."""
    rng = np.random.default_rng(11)
    # (a) 300 000 cells x 64 genes, ~6 stored entries per cell
    n, G = 300_000, 64
    lens = rng.integers(0, 13, n)
    ip = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    ix = np.concatenate([np.sort(rng.choice(G, l, replace=False)) for l in lens[:2000]] +
                        [np.empty(0, dtype=np.int64)]).astype(np.int32)
    # cheap generation for the bulk: the first 2000 rows' pattern repeats (rows stay canonical)
    reps = -(-n // 2000)
    lens2 = np.tile(lens[:2000], reps)[:n]
    ip = np.concatenate([[0], np.cumsum(lens2)]).astype(np.int64)
    ix = np.tile(ix, reps)[: ip[-1]].astype(np.int32)
    dl = (0.3 + 3.0 * rng.random(ip[-1])).astype(np.float32)
    _check(ip, ix, dl, G)
    # (b) 1 200 cells x 4 500 genes (18 x 36 tiles, ragged last tiles)
    n, G = 1200, 4500
    dense = (rng.random((n, G)) < 0.03) * (0.3 + 3.0 * rng.random((n, G)))
    r, c = np.nonzero(dense)
    ip = np.concatenate([[0], np.cumsum(np.bincount(r, minlength=n))]).astype(np.int64)
    _check(ip, c.astype(np.int32), dense[r, c].astype(np.float32), G)
