"""GPU parity of SURVEY.md 8(f) NEXT-1 (filter masks, CSR row / column subsetting) against the
CPU oracle: masks and the subset CSR are integer / copied-value work => bit-exact."""
import numpy as np
import pytest
import torch

from oracle import oracle_np as O
from paper_2603_02402_b200 import synth
import parity_util as U

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2603_02402_b200 import build, binding
    build.build()
    binding.lib()
    assert torch.cuda.is_available()


CASES = [(1, 1, 0, 3.0, (), ()), (3, 7, 1, 2.0, (1,), (2,)), (257, 1031, 2, 0.7, (0, 100, 256), (0, 1030)),
         (2500, 4099, 3, 0.4, (17,), (5, 6, 7)), (33, 36000, 5, 0.6, (32,), ())]


def _check_subset(indptr, indices, data, G, kr, kc):
    from paper_2603_02402_b200 import binding as B
    X = U.to_dev(indptr, indices, data, G)
    ip_o, ix_o, dt_o, g_o = O.subset_csr(indptr, indices, data, G,
                                         np.ones(len(indptr) - 1, bool) if kr is None else kr,
                                         np.ones(G, bool) if kc is None else kc)
    Y, g_g = B.rsc_subset_csr(X, None if kr is None else torch.as_tensor(kr.astype(np.uint8)).cuda(),
                              None if kc is None else torch.as_tensor(kc.astype(np.uint8)).cuda())
    torch.cuda.synchronize()
    assert g_g == g_o
    U.assert_int_equal(Y.indptr, ip_o, "subset indptr")
    U.assert_int_equal(Y.indices, ix_o, "subset indices")
    assert np.array_equal(U.np_(Y.data), dt_o), "subset data"
    assert np.array_equal(U.np_(X.data), data) and np.array_equal(U.np_(X.indices), indices)   # input untouched


@pytest.mark.parametrize("n,G,seed,depth,er,eg", CASES)
def test_subset_csr(n, G, seed, depth, er, eg):
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    rng = np.random.default_rng(100 + seed)
    for pr, pc in ((0.6, 0.5), (1.0, 1.0), (0.0, 0.7), (0.7, 0.0), (1.0, 0.1), (0.05, 1.0)):
        _check_subset(indptr, indices, data, G, rng.random(n) < pr, rng.random(G) < pc)
    _check_subset(indptr, indices, data, G, None, None)            # NULL masks: the identity
    _check_subset(indptr, indices, data, G, None, rng.random(G) < 0.3)


@pytest.mark.parametrize("n,G,seed,depth,er,eg", CASES[2:])
def test_filter_masks_then_subset_then_chain(n, G, seed, depth, er, eg):
    """QC -> masks -> subset, all on the device, equals the oracle's; the preprocessing of the
    filtered matrix equals the oracle's on the oracle-filtered matrix (same arrays)."""
    from paper_2603_02402_b200 import binding as B
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    flags = np.zeros(G, np.uint8); flags[:13] = 1
    X = U.to_dev(indptr, indices, data, G)
    q = B.rsc_qc_metrics(X, torch.as_tensor(flags).cuda())
    q_o = O.qc_metrics(indptr, indices, data, G, flags)
    for thr in (dict(), dict(min_genes=5, min_counts=8, max_pct_flag=20.0, min_cells=2, min_gene_counts=3),
                dict(min_genes=10**6), dict(max_pct_flag=0.0)):
        ck, gk = B.rsc_filter_masks(q, **thr)
        ck_o, gk_o = O.filter_masks(q_o, **thr)
        U.assert_int_equal(ck, ck_o, f"cell mask {thr}")
        U.assert_int_equal(gk, gk_o, f"gene mask {thr}")
        Y, g2 = B.rsc_subset_csr(X, ck, gk)
        ip_o, ix_o, dt_o, g_o = O.subset_csr(indptr, indices, data, G, ck_o, gk_o)
        assert g2 == g_o
        U.assert_int_equal(Y.indptr, ip_o, "indptr"); U.assert_int_equal(Y.indices, ix_o, "indices")
        assert np.array_equal(U.np_(Y.data), dt_o)
        if g2 > 0 and Y.n_rows > 1 and Y.nnz > 0:
            q2 = B.rsc_qc_metrics(Y)
            out = B.rsc_normalize_log1p_moments(Y, 1e4, q2["cell_total_i64"], q2["gene_n_cells"], 1, 1)
            mo, vo, _, _ = O.gene_moments(ip_o, ix_o, U.np_(Y.data), g_o, 0, 1)
            U.assert_moments_close(out["mean_log"], out["var_log"], mo, vo, "moments of the filtered matrix")


def test_subset_full_size_invariants():
    """cfg2 at full size: HVG-style column subsetting + cell filter; sampled rows against the
    oracle, sizes against the masks."""
    from paper_2603_02402_b200 import binding as B, Csr
    cfg = synth.CONFIGS[2]
    indptr, indices, data = synth.make_csr(cfg, "cuda")
    X = Csr(indptr, indices, data, cfg.n_genes)
    q = B.rsc_qc_metrics(X, synth.gene_flags(cfg, "cuda"))
    ck, gk = B.rsc_filter_masks(q, min_genes=1500, min_cells=1000)
    Y, g2 = B.rsc_subset_csr(X, ck, gk)
    torch.cuda.synchronize()
    assert g2 == int(gk.sum()) and Y.n_rows == int(ck.sum())
    assert int(Y.indptr[-1]) == Y.nnz and bool((Y.indices >= 0).all()) and bool((Y.indices < g2).all())
    rng = np.random.default_rng(0)
    kept = torch.nonzero(ck).flatten().cpu().numpy()
    rows = np.unique(np.concatenate([rng.choice(kept, 64), kept[:2], kept[-2:]]))
    ip, ix, (dt,), _ = U.extract_rows(indptr, indices, [data], rows)
    ip_o, ix_o, dt_o, _ = O.subset_csr(ip, ix, dt, cfg.n_genes, np.ones(len(rows), bool), U.np_(gk).astype(bool))
    rank = np.cumsum(U.np_(ck).astype(np.int64)) - 1
    ipy, ixy, (dty,), _ = U.extract_rows(Y.indptr, Y.indices, [Y.data], rank[rows])
    assert np.array_equal(ipy, ip_o) and np.array_equal(ixy, ix_o) and np.array_equal(dty, dt_o)
