"""The C / OpenMP oracle twin (oracle/oracle_c.c) against oracle_np, element by element: integer
outputs equal, float32 outputs bit-equal (same float64 expression, one rounding), float64 sums
within 1e-12 relative (only the summation order differs).  oracle_np itself is pinned in
tests/test_oracle_*.py; this file makes the twin inherit those pins."""
import numpy as np
import pytest

from oracle import oracle_c as OC
from oracle import oracle_np as O
from paper_2603_02402_b200 import synth

CASES = [(1, 7, 0, 0.5, (), ()), (37, 200, 1, 0.3, (3,), (5, 6)), (300, 1500, 2, 0.2, (0, 7, 299), (40, 1499)),
         (900, 3000, 3, 0.1, (), ())]


@pytest.mark.parametrize("n,G,seed,depth,er,eg", CASES)
@pytest.mark.parametrize("threads", [1, 4])
def test_c_twin_matches_numpy_oracle(n, G, seed, depth, er, eg, threads):
    OC.set_num_threads(threads)
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    flags = np.zeros(G, np.uint8); flags[: min(G, 5)] = 1
    q, qc = O.qc_metrics(indptr, indices, data, G, flags), OC.qc_metrics(indptr, indices, data, G, flags)
    for k in ("cell_total_i64", "cell_n_genes", "cell_flag_total_i64", "gene_n_cells", "gene_total_i64"):
        assert q[k].dtype == qc[k].dtype and np.array_equal(q[k], qc[k]), k
    assert np.array_equal(q["cell_flag_pct"], qc["cell_flag_pct"], equal_nan=True)
    xn_o, _ = O.normalize_total(indptr, data, 1e4, q["cell_total_i64"])
    xl_o = O.log1p(xn_o)
    xn_c, xl_c = OC.normalize_log1p(indptr, data, 1e4, q["cell_total_i64"])
    assert np.array_equal(xn_o, xn_c) and np.array_equal(xl_o, xl_c)
    for tr, arr in ((0, xl_o), (1, xl_o), (0, xn_o)):
        mo, vo, s1o, s2o = O.gene_moments(indptr, indices, arr, G, tr, 1)
        mc, vc, s1c, s2c = OC.gene_moments(indptr, indices, arr, G, tr, 1)
        np.testing.assert_allclose(s1c, s1o, rtol=1e-12, atol=0)
        np.testing.assert_allclose(s2c, s2o, rtol=1e-12, atol=0)
        np.testing.assert_allclose(mc, mo, rtol=1e-12, atol=0)
        np.testing.assert_allclose(vc, vo, rtol=1e-11, atol=1e-300)


def test_c_twin_row_chunks_accumulate():
    """Walking the matrix in row chunks and accumulating the per-gene outputs gives the one-shot
    result (this is how the full-size GPU parity tests and bench.py's CPU baseline use it)."""
    n, G = 500, 800
    indptr, indices, data, _ = synth.small_nb_csr(n, G, 5, 0.2, empty_rows=(4, 130), empty_genes=(9,))
    whole = OC.qc_metrics(indptr, indices, data, G, None)
    gn, gt = np.zeros(G, np.int64), np.zeros(G, np.int64)
    s = (np.zeros(G), np.zeros(G), np.zeros(G))
    tot = []
    for a in range(0, n, 128):
        b = min(n, a + 128)
        ip = indptr[a:b + 1] - indptr[a]
        sl = slice(int(indptr[a]), int(indptr[b]))
        part = OC.qc_metrics(ip, indices[sl], data[sl], G, None, gene_acc=(gn, gt))
        tot.append(part["cell_total_i64"])
        OC.gene_sums(ip, indices[sl], data[sl], G, 0, acc=s)
    assert np.array_equal(np.concatenate(tot), whole["cell_total_i64"])
    assert np.array_equal(gn.astype(np.int32), whole["gene_n_cells"]) and np.array_equal(gt, whole["gene_total_i64"])
    s1, s2, st = OC.gene_sums(indptr, indices, data, G, 0)
    np.testing.assert_allclose(s[0], s1, rtol=1e-13); np.testing.assert_allclose(s[1], s2, rtol=1e-13)
    assert np.array_equal(s[2], st)


def test_c_chain_equals_numpy_chain():
    cfg = synth.scaled(synth.CONFIGS[1], 300)
    indptr, indices, data = (t.numpy() for t in synth.make_csr(cfg, "cpu"))
    flags = synth.gene_flags(cfg, "cpu").numpy()
    a = O.preprocess_chain(indptr, indices, data, cfg.n_genes, flags, cfg.target_sum, 200, cfg.n_bins)
    b = OC.preprocess_chain(indptr, indices, data, cfg.n_genes, flags, cfg.target_sum, 200, cfg.n_bins)
    assert np.array_equal(a["x_log"], b["x_log"]) and np.array_equal(a["x_norm"], b["x_norm"])
    np.testing.assert_allclose(b["mean_lin"], a["mean_lin"], rtol=1e-12)
    np.testing.assert_allclose(b["var_lin"], a["var_lin"], rtol=1e-11)
    assert np.array_equal(a["hvg"]["mask"], b["hvg"]["mask"])
    assert OC.num_threads() >= 1
