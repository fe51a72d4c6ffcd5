"""GPU parity of the single-pass chain (csrc/single.cu, option "single_pass"): QC + normalise +
log1p + log-scale moments in ONE pass over the matrix by pairs of CTAs that exchange the rows'
partial totals through distributed shared memory ("theoretical single
pass").  Checked against the oracle (integers exact, x'' 1e-5, moments 1e-9
on the x'' the GPU wrote) and, bit for bit, against the default two-kernel chain.
"""
import numpy as np
import pytest
import torch

from oracle import oracle_np as O
from paper_2603_02402_b200 import synth
import parity_util as U

pytestmark = pytest.mark.gpu

INT_KEYS = ("cell_total_i64", "cell_n_genes", "cell_flag_total_i64", "gene_n_cells", "gene_total_i64")


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2603_02402_b200 import build, binding
    build.build()
    binding.lib()


@pytest.fixture
def single_pass():
    from paper_2603_02402_b200 import binding as B
    B.rsc_set_option("single_pass", 1)
    yield
    B.rsc_set_option("single_pass", 0)
    B.rsc_set_option("fused_row_budget", 256)
    B.rsc_set_option("flush_all", 0)
    B.rsc_set_option("grid_ctas", 0)


def _chain(X, flags, s, n_top, n_bins=20):
    """rsc_preprocess, log-scale moments only; returns (outputs, kernels launched)."""
    from paper_2603_02402_b200 import binding as B
    before = B.rsc_kernel_launch_count()
    out = B.rsc_preprocess(X, flags, s, n_top, n_bins, which_moments=1, hvg_on_linear=False)
    torch.cuda.synchronize()
    return out, B.rsc_kernel_launch_count() - before


def _both(indptr, indices, data, G, flags_np, s, n_top):
    """Runs the default chain and the single-pass chain on copies of one matrix."""
    from paper_2603_02402_b200 import binding as B
    fl = None if flags_np is None else torch.as_tensor(flags_np).cuda()
    X0 = U.to_dev(indptr, indices, data, G)
    X1 = U.clone(X0)
    B.rsc_set_option("single_pass", 0)
    o0, l0 = _chain(X0, fl, s, n_top)
    o0 = {k: v.clone() for k, v in o0.items() if torch.is_tensor(v)}
    B.rsc_set_option("single_pass", 1)
    o1, l1 = _chain(X1, fl, s, n_top)
    return X0, o0, l0, X1, o1, l1


def _assert_same(X0, o0, X1, o1, tag):
    for k in INT_KEYS + ("hvg_bin", "hvg_mask", "hvg_count"):
        assert torch.equal(o0[k], o1[k]), f"{tag}: {k} differs between the two chains"
    assert torch.equal(X0.data, X1.data), f"{tag}: x'' differs"
    for k in ("cell_total_f32", "cell_flag_pct"):
        assert np.array_equal(U.np_(o0[k]), U.np_(o1[k]), equal_nan=True), f"{tag}: {k}"
    # exact integer accumulators on both sides; the two plans may place the window of the squares
    # differently (all cells vs a sample), which moves S2 by <= 2^-39 relative per entry
    np.testing.assert_allclose(U.np_(o1["mean_log"]), U.np_(o0["mean_log"]), rtol=1e-13, atol=0)
    np.testing.assert_allclose(U.np_(o1["var_log"]), U.np_(o0["var_log"]), rtol=1e-9, atol=1e-300)


def test_config1_against_the_oracle(single_pass):
    from paper_2603_02402_b200 import Csr
    cfg = synth.CONFIGS[1]
    indptr, indices, data = synth.make_csr(cfg, "cuda")
    flags = synth.gene_flags(cfg, "cuda")
    raw = data.clone()
    X = Csr(indptr, indices, data, cfg.n_genes)
    out, launches = _chain(X, flags, cfg.target_sum, cfg.n_top, cfg.n_bins)
    ip, ix, rw = U.np_(indptr), U.np_(indices), U.np_(raw)
    q = O.qc_metrics(ip, ix, rw, cfg.n_genes, U.np_(flags))
    for k in INT_KEYS:
        U.assert_int_equal(out[k], q[k], k)
    U.assert_f32_close(out["cell_flag_pct"], q["cell_flag_pct"], "pct")
    U.assert_f32_close(out["cell_total_f32"], q["cell_total_f32"], "total f32")
    xl_o = O.log1p(O.normalize_total(ip, rw, cfg.target_sum)[0])
    U.assert_f32_close(X.data, xl_o, "x''")
    mo, vo, _, _ = O.gene_moments(ip, ix, U.np_(X.data), cfg.n_genes, 0, 1)
    U.assert_moments_close(out["mean_log"], out["var_log"], mo, vo, "log moments")
    ref = O.hvg_select(U.np_(out["mean_log"]), U.np_(out["var_log"]), cfg.n_top, cfg.n_bins)
    g = dict(mean_t=out["hvg_mean_t"], disp=out["hvg_disp"], disp_norm=out["hvg_disp_norm"],
             bin=out["hvg_bin"], mask=out["hvg_mask"], indices=out["hvg_indices"], count=out["hvg_count"])
    U.assert_hvg_matches(g, ref, cfg.n_top, "hvg", strict=False)
    # the single-pass kernel really ran: its chain launches one kernel more than the default one
    from paper_2603_02402_b200 import binding as B
    B.rsc_set_option("single_pass", 0)
    X.data.copy_(raw)
    _, launches_default = _chain(X, flags, cfg.target_sum, cfg.n_top, cfg.n_bins)
    assert launches == launches_default + 1


@pytest.mark.parametrize("n,G,seed,depth", [(2, 600, 0, 1.0), (3, 513, 1, 1.0), (45, 777, 2, 3.0),
                                            (700, 2100, 3, 0.5), (3000, 18000, 4, 0.15),
                                            (1500, 32768, 5, 0.1)])
def test_equals_the_two_kernel_chain(single_pass, n, G, seed, depth):
    er = (0, n - 1) if n > 40 else ()
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=(7, G - 1))
    flags = np.zeros(G, np.uint8)
    flags[:37] = 1
    flags[G // 2 - 3:G // 2 + 3] = 1                        # flagged genes on both sides of the boundary
    X0, o0, l0, X1, o1, l1 = _both(indptr, indices, data, G, flags, 1e4, min(200, G // 4))
    assert l1 == l0 + 1, "the single-pass kernel did not run"
    _assert_same(X0, o0, X1, o1, f"n={n} G={G}")
    q = O.qc_metrics(indptr, indices, data, G, flags)
    for k in INT_KEYS:
        U.assert_int_equal(o1[k], q[k], k)


def test_special_values_and_flush_paths(single_pass):
    """Counts beyond the shared table's fields (> 4), beyond the packed row sums (> 511), explicit
    zeros, fractions, negative values; every table check moves every gene (flush_all), checks
    every 8 rows, an odd grid request."""
    from paper_2603_02402_b200 import binding as B
    n, G = 900, 3000
    indptr, indices, data, _ = synth.small_nb_csr(n, G, 21, 2.0, empty_rows=(5, 6, 899))
    data = data.copy()
    rng = np.random.default_rng(21)
    pick = rng.permutation(len(data))
    data[pick[:300]] = 0.0
    data[pick[300:600]] = rng.integers(5, 512, 300).astype(np.float32)
    data[pick[600:700]] = rng.integers(512, 100000, 100).astype(np.float32)
    data[pick[700:760]] = 0.5
    data[pick[760:800]] = -3.0
    flags = (rng.random(G) < 0.05).astype(np.uint8)
    for opts in ({}, {"flush_all": 1, "fused_row_budget": 8, "grid_ctas": 7}):
        for k, v in opts.items():
            B.rsc_set_option(k, v)
        X0, o0, l0, X1, o1, l1 = _both(indptr, indices, data, G, flags, 1e4, 300)
        assert l1 == l0 + 1
        q = O.qc_metrics(indptr, indices, data, G, flags)
        for k in INT_KEYS:
            U.assert_int_equal(o1[k], q[k], f"{k} {opts}")
        # x'' and the integer sums must agree with the default chain; negative x' makes moments of
        # NaN / huge values order-dependent in the global double sums, so compare them loosely
        assert torch.equal(torch.nan_to_num(X0.data, nan=-1.0), torch.nan_to_num(X1.data, nan=-1.0))
        m0, m1 = U.np_(o0["mean_log"]), U.np_(o1["mean_log"])
        ok = np.isfinite(m0)
        assert np.array_equal(ok, np.isfinite(m1))
        np.testing.assert_allclose(m1[ok], m0[ok], rtol=1e-9)


def test_falls_back_when_it_cannot_serve(single_pass):
    """More genes than two CTAs hold, or the linear-scale set: the default chain runs (same
    number of launches as with the option off)."""
    n, G = 300, 33000
    indptr, indices, data, _ = synth.small_nb_csr(n, G, 8, 0.1)
    X0, o0, l0, X1, o1, l1 = _both(indptr, indices, data, G, None, 1e4, 500)
    assert l1 == l0
    _assert_same(X0, o0, X1, o1, "fallback")
