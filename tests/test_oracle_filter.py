"""Pins for the NEXT-1 oracle functions (filter masks, CSR row / column subsetting): dense
brute force, scipy.sparse fancy indexing, identity and drop-all cases, nnz bookkeeping."""
import numpy as np
import pytest
import scipy.sparse as sp

from oracle import oracle_np as O
from paper_2603_02402_b200 import synth

CASES = [(1, 1, 0, 3.0), (7, 5, 1, 2.0), (120, 333, 2, 0.8), (400, 2100, 3, 0.3)]


@pytest.mark.parametrize("n,G,seed,depth", CASES)
def test_subset_csr_dense_and_scipy(n, G, seed, depth):
    indptr, indices, data, dense = synth.small_nb_csr(n, G, seed, depth, empty_rows=(0,) if n > 3 else ())
    rng = np.random.default_rng(seed)
    for pr, pc in ((0.6, 0.5), (1.0, 1.0), (0.0, 0.7), (0.7, 0.0), (1.0, 0.1)):
        kr = rng.random(n) < pr
        kc = rng.random(G) < pc
        ip, ix, dt, g2 = O.subset_csr(indptr, indices, data, G, kr, kc)
        want = dense[kr][:, kc]
        assert g2 == int(kc.sum()) and len(ip) == int(kr.sum()) + 1 and ip[0] == 0 and ip[-1] == len(ix) == len(dt)
        got = np.zeros(want.shape)
        for r in range(len(ip) - 1):
            got[r, ix[ip[r]:ip[r + 1]]] = dt[ip[r]:ip[r + 1]]
            assert np.all(np.diff(ix[ip[r]:ip[r + 1]]) > 0)          # order kept => still ascending
        assert np.array_equal(got, want)
        m = sp.csr_matrix((data, indices, indptr), shape=(n, G))[np.nonzero(kr)[0]][:, np.nonzero(kc)[0]]
        m.sort_indices()
        assert np.array_equal(m.indptr, ip) and np.array_equal(m.indices, ix) and np.array_equal(m.data, dt)
        assert len(ix) == int((want != 0).sum())                    # generator stores no zeros


def test_subset_keeps_explicit_zeros_and_identity():
    indptr = np.array([0, 3, 3, 5], np.int64)
    indices = np.array([0, 2, 4, 1, 4], np.int32)
    data = np.array([1, 0, 2, 3, 0], np.float32)                   # explicit zeros stay stored
    ip, ix, dt, g2 = O.subset_csr(indptr, indices, data, 5, [1, 1, 1], [1, 1, 1, 1, 1])
    assert np.array_equal(ip, indptr) and np.array_equal(ix, indices) and np.array_equal(dt, data) and g2 == 5
    ip, ix, dt, g2 = O.subset_csr(indptr, indices, data, 5, [1, 0, 1], [0, 1, 1, 0, 1])
    assert ip.tolist() == [0, 2, 4] and ix.tolist() == [1, 2, 0, 2] and dt.tolist() == [0, 2, 3, 0] and g2 == 3


def test_filter_masks_thresholds():
    indptr, indices, data, dense = synth.small_nb_csr(200, 500, 5, 0.5, empty_rows=(3,), empty_genes=(4,))
    flags = np.zeros(500, np.uint8); flags[:13] = 1
    q = O.qc_metrics(indptr, indices, data, 500, flags)
    c, g = O.filter_masks(q)                                       # no thresholds: everything stays
    assert c.all() and g.all()
    c, g = O.filter_masks(q, min_genes=20, min_counts=30, max_pct_flag=10.0, min_cells=3, min_gene_counts=5)
    ng, tot = (dense != 0).sum(1), dense.sum(1)
    pct = 100.0 * dense[:, :13].sum(1) / np.where(tot > 0, tot, np.nan)
    want_c = (ng >= 20) & (tot >= 30) & (np.nan_to_num(pct, nan=np.inf) <= 10.0)
    want_g = ((dense != 0).sum(0) >= 3) & (dense.sum(0) >= 5)
    assert np.array_equal(c.astype(bool), want_c) and np.array_equal(g.astype(bool), want_g)
    assert not c[3] and not g[4]                                   # the empty cell / gene go
