"""GPU parity of SURVEY 8(f) NEXT-4: rsc_hvg_select_cell_ranger and rsc_hvg_merge_batches against
oracle_np (bit-exact: every order statistic is an exact selection and the arithmetic uses the
same separate multiply / add as the oracle), and the per-batch workflow over row ranges."""
import numpy as np
import pytest
import torch

from oracle import oracle_np as O
from paper_2603_02402_b200 import Csr, binding as B, synth

pytestmark = pytest.mark.gpu


def _moments(G, seed, zeros=0, ties=False):
    rng = np.random.default_rng(seed)
    mean = np.exp(rng.normal(-1.0, 1.5, G))
    var = mean * np.exp(rng.normal(0.3, 0.6, G))
    if ties:
        mean = np.round(mean, 1); var = np.round(var, 1)
    if zeros:
        idx = rng.choice(G, zeros, replace=False)
        mean[idx] = 0.0; var[idx] = 0.0
    return mean, var


def _check_cr(mean, var, n_top):
    r = O.hvg_cell_ranger(mean, var, n_top)
    g = B.rsc_hvg_select_cell_ranger(torch.from_numpy(mean).cuda(), torch.from_numpy(var).cuda(), n_top)
    torch.cuda.synchronize()
    assert np.array_equal(g["disp"].cpu().numpy(), r["disp"])
    assert np.array_equal(g["bin"].cpu().numpy(), r["bin"])
    np.testing.assert_array_equal(g["disp_norm"].cpu().numpy(), r["disp_norm"])     # NaN == NaN here
    assert np.array_equal(g["mask"].cpu().numpy().astype(bool), r["mask"])
    c = int(g["count"][0])
    assert c == r["count"]
    assert np.array_equal(g["indices"].cpu().numpy()[:c], r["indices"])


@pytest.mark.parametrize("G,seed,zeros,ties,n_top", [(21, 0, 0, False, 3), (400, 1, 0, False, 40), (3000, 2, 200, False, 300),
                                                      (30000, 3, 1500, False, 4000), (36000, 4, 0, True, 3000),
                                                      (500, 5, 350, True, 50), (64, 6, 0, False, 1000)])
def test_cell_ranger_matches_oracle(G, seed, zeros, ties, n_top):
    mean, var = _moments(G, seed, zeros, ties)
    _check_cr(mean, var, n_top)


def test_cell_ranger_fixture_on_device():
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "hvg_cell_ranger_tiny.txt"))
            if l.strip() and l[0] != "#"]
    mean = np.array([float(r[1]) for r in rows]); var = np.array([float(r[2]) for r in rows])
    g = B.rsc_hvg_select_cell_ranger(torch.from_numpy(mean).cuda(), torch.from_numpy(var).cuda(), 2)
    assert g["mask"].cpu().numpy().tolist() == [int(r[6]) for r in rows]
    np.testing.assert_array_equal(g["disp_norm"].cpu().numpy(), np.array([float(r[5]) for r in rows]))


@pytest.mark.parametrize("Bn,G,seed,n_top", [(1, 300, 0, 30), (3, 5000, 1, 600), (8, 30000, 2, 4000), (2, 40, 3, 100)])
def test_merge_batches_matches_oracle(Bn, G, seed, n_top):
    rng = np.random.default_rng(seed)
    z = rng.normal(0, 1, (Bn, G))
    z[rng.random((Bn, G)) < 0.15] = np.nan
    if seed == 2:
        z = np.round(z, 1)                                   # ties at the cutoff
    masks = np.zeros((Bn, G), dtype=np.uint8)
    for b in range(Bn):
        zb = np.where(np.isnan(z[b]), -np.inf, z[b])
        masks[b, np.argsort(-zb)[: min(n_top, G)]] = 1
    r = O.hvg_merge_batches(masks, z, n_top)
    g = B.rsc_hvg_merge_batches(torch.from_numpy(masks).cuda(), torch.from_numpy(z).cuda(), n_top)
    torch.cuda.synchronize()
    assert np.array_equal(g["nbatches"].cpu().numpy(), r["nbatches"])
    np.testing.assert_array_equal(g["disp_norm_mean"].cpu().numpy(), r["disp_norm_mean"])
    assert np.array_equal(g["mask"].cpu().numpy().astype(bool), r["mask"])
    c = int(g["count"][0])
    assert c == r["count"] and np.array_equal(g["indices"].cpu().numpy()[:c], r["indices"])


def test_merge_all_nan_level_tail():
    masks = np.zeros((2, 6), dtype=np.uint8)
    z = np.full((2, 6), np.nan); z[:, 4] = 1.0
    r = O.hvg_merge_batches(masks, z, 3)
    g = B.rsc_hvg_merge_batches(torch.from_numpy(masks).cuda(), torch.from_numpy(z).cuda(), 3)
    assert np.array_equal(g["mask"].cpu().numpy().astype(bool), r["mask"])


@pytest.mark.parametrize("flavor", ["seurat", "cell_ranger"])
def test_batched_workflow(flavor):
    cfg = synth.scaled(synth.CONFIGS[2], 6000)
    indptr, indices, data = synth.make_csr(cfg, "cuda")
    flags = synth.gene_flags(cfg, "cuda")
    raw = data.clone()
    X = Csr(indptr, indices, data, cfg.n_genes)
    offs = [0, 1500, 3700, 6000]
    out = B.rsc_hvg_select_batched(X, offs, flags, cfg.target_sum, 1200, cfg.n_bins, flavor=flavor)
    torch.cuda.synchronize()
    # the merge against the oracle, fed with the device's per-batch outputs
    r = O.hvg_merge_batches(out["batch_masks"].cpu().numpy(), out["batch_disp_norm"].cpu().numpy(), 1200)
    assert np.array_equal(out["mask"].cpu().numpy().astype(bool), r["mask"])
    assert np.array_equal(out["nbatches"].cpu().numpy(), r["nbatches"])
    # every batch's selection against the oracle on that batch's (device) linear-scale moments
    for b, o in enumerate(out["per_batch"]):
        m, v = o["mean_lin"].cpu().numpy(), o["var_lin"].cpu().numpy()
        if flavor == "cell_ranger":
            want = O.hvg_cell_ranger(m, v, 1200)
        else:
            want = O.hvg_select(m, v, 1200, cfg.n_bins)
        assert np.array_equal(out["batch_masks"][b].cpu().numpy().astype(bool), want["mask"].astype(bool))
    # in-place chain per row range == the chain on the whole matrix (rows are independent)
    xa = X.data.clone()
    X.data.copy_(raw)
    B.rsc_preprocess(X, flags, cfg.target_sum, 1200, cfg.n_bins)
    assert torch.equal(xa, X.data)
