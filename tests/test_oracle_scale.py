"""Pins for the NEXT-3 oracle function scale_dense: numpy on the dense matrix, column mean 0 /
sd 1 when unclipped, zero-variance genes, clip bounds, zero_center = False."""
import numpy as np
import pytest

from oracle import oracle_np as O
from paper_2603_02402_b200 import synth


@pytest.mark.parametrize("n,G,seed,depth", [(50, 40, 0, 2.0), (300, 120, 1, 0.8)])
def test_scale_dense_against_numpy(n, G, seed, depth):
    indptr, indices, data, dense = synth.small_nb_csr(n, G, seed, depth, empty_genes=(3,))
    xl = np.log1p(dense)
    ip, ix = indptr, indices
    dl = np.log1p(data.astype(np.float64)).astype(np.float32)
    dense_l = np.zeros_like(dense); r = np.repeat(np.arange(n), np.diff(indptr)); dense_l[r, indices] = dl
    mean, var, _, _ = O.gene_moments(ip, ix, dl, G, 0, 1)
    y = O.scale_dense(ip, ix, dl, G, mean, var)
    sd = dense_l.std(axis=0, ddof=1); sd[sd == 0] = 1
    want = (dense_l - dense_l.mean(axis=0)) / sd
    np.testing.assert_allclose(y, want.astype(np.float32), rtol=2e-6, atol=2e-6)
    live = dense_l.std(axis=0) > 0
    np.testing.assert_allclose(y[:, live].mean(axis=0), 0, atol=1e-5)
    np.testing.assert_allclose(y[:, live].std(axis=0, ddof=1), 1, rtol=1e-5)
    assert np.all(y[:, 3] == 0)                                     # empty gene: (0 - 0) / 1
    yc = O.scale_dense(ip, ix, dl, G, mean, var, max_value=1.5)
    assert yc.max() <= 1.5 and yc.min() >= -1.5 and np.array_equal(yc, np.clip(y, -1.5, 1.5))
    yn = O.scale_dense(ip, ix, dl, G, mean, var, max_value=2.0, zero_center=False)
    assert np.all(yn[dense_l == 0] == 0) and yn.max() <= 2.0
    np.testing.assert_allclose(yn, np.minimum(dense_l / sd, 2.0).astype(np.float32), rtol=2e-6)
