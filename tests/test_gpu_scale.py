"""GPU parity of SURVEY.md 8(f) NEXT-3 (first half), rsc_scale_dense, against the CPU oracle:
float32 z-scores within 1e-5 relative (plus 1e-6 absolute around zero)."""
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


def _close(got, want, name):
    got = U.np_(got).astype(np.float64); want = want.astype(np.float64)
    err = np.abs(got - want)
    assert np.all(err <= 1e-5 * np.abs(want) + 1e-6), f"{name}: max err {err.max():.3e}"


@pytest.mark.parametrize("n,G,seed,depth", [(1, 1, 0, 3.0), (3, 7, 1, 2.0), (257, 1031, 2, 0.7), (700, 4000, 3, 0.4),
                                            (64, 2049, 4, 1.0)])
def test_scale_dense(n, G, seed, depth):
    from paper_2603_02402_b200 import binding as B
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=(0,) if n > 2 else (),
                                                  empty_genes=(2,) if G > 3 else ())
    dl = np.log1p(data.astype(np.float64)).astype(np.float32)
    ddof = 1 if n > 1 else 0
    mean, var, _, _ = O.gene_moments(indptr, indices, dl, G, 0, ddof)
    X = U.to_dev(indptr, indices, dl, G)
    m, v = torch.as_tensor(mean).cuda(), torch.as_tensor(var).cuda()
    for mv, zc in ((None, True), (10.0, True), (0.5, True), (None, False), (1.0, False)):
        y = B.rsc_scale_dense(X, m, v, mv, zc)
        torch.cuda.synchronize()
        _close(y, O.scale_dense(indptr, indices, dl, G, mean, var, mv, zc), f"scale mv={mv} zc={zc}")
    assert np.array_equal(U.np_(X.data), dl)                       # input untouched


def test_chain_filter_hvg_subset_scale():
    """raw counts -> QC -> filter -> normalise+log1p+moments -> HVG -> column subset -> scale, all on
    the device; the scaled HVG matrix equals the oracle's on the same x'' / moments."""
    from paper_2603_02402_b200 import binding as B
    cfg = synth.scaled(synth.CONFIGS[1], 2000)
    indptr, indices, data = synth.make_csr(cfg, "cuda")
    from paper_2603_02402_b200 import Csr
    X = Csr(indptr, indices, data, cfg.n_genes)
    q = B.rsc_qc_metrics(X, synth.gene_flags(cfg, "cuda"))
    ck, gk = B.rsc_filter_masks(q, min_genes=100, min_cells=3)
    Y, g2 = B.rsc_subset_csr(X, ck, gk)
    q2 = B.rsc_qc_metrics(Y)
    mom = B.rsc_normalize_log1p_moments(Y, cfg.target_sum, q2["cell_total_i64"], q2["gene_n_cells"], 1, 1)
    h = B.rsc_hvg_select(mom["mean_log"], mom["var_log"], 300, cfg.n_bins, 1)
    Z, g3 = B.rsc_subset_csr(Y, None, h["mask"])
    assert g3 == int(h["count"][0]) >= 300
    sel = torch.nonzero(h["mask"]).flatten()
    y = B.rsc_scale_dense(Z, mom["mean_log"][sel].contiguous(), mom["var_log"][sel].contiguous(), 10.0, True)
    torch.cuda.synchronize()
    want = O.scale_dense(U.np_(Z.indptr), U.np_(Z.indices), U.np_(Z.data), g3, U.np_(mom["mean_log"][sel]),
                         U.np_(mom["var_log"][sel]), 10.0, True)
    _close(y, want, "scaled HVG matrix")
    live = U.np_(mom["var_log"][sel]) > 0
    yy = U.np_(y).astype(np.float64)[:, live]
    unclipped = np.abs(yy).max(axis=0) < 10.0                      # columns the clip did not touch
    np.testing.assert_allclose(yy[:, unclipped].mean(axis=0), 0, atol=1e-4)


@pytest.mark.parametrize("G,seed", [(1, 0), (50, 1), (4099, 2), (36000, 3)])
def test_hvg_cutoffs(G, seed):
    """NEXT-4 (part): threshold-based selection on the device == the oracle's, bit-exact."""
    from paper_2603_02402_b200 import binding as B
    rng = np.random.default_rng(seed)
    mean = np.exp(rng.normal(-3, 2, G)); var = mean * np.exp(rng.normal(0.2, 0.6, G))
    mean[rng.random(G) < 0.1] = 0.0
    h = B.rsc_hvg_select(torch.as_tensor(mean).cuda(), torch.as_tensor(var).cuda(), max(1, G // 10), 20, 1)
    m, z = U.np_(h["mean_t"]), U.np_(h["disp_norm"])
    for win in ((0.0125, 3.0, 0.5, np.inf), (-np.inf, np.inf, -np.inf, np.inf), (0.05, 0.05, 0.0, 1.0),
                (0.0, 10.0, -0.25, 2.0)):
        o = O.hvg_cutoffs(m, z, *win)
        g = B.rsc_hvg_cutoffs(h["mean_t"], h["disp_norm"], *win)
        torch.cuda.synchronize()
        c = int(U.np_(g["count"])[0])
        assert c == o["count"]
        U.assert_int_equal(g["mask"], o["mask"], f"cutoff mask {win}")
        assert np.array_equal(U.np_(g["indices"])[:c], o["indices"])
