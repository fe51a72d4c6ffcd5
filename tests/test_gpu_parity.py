"""GPU parity: every C-ABI entry point against the CPU oracle on the same seeded inputs.

Integers bit-exact; float32 values within 1e-5 relative; fp64 moments within 1e-9 when both
sides read bit-identical float32 inputs; HVG set identical up to ties at the cutoff
(BASELINE.json north_star).
"""
import numpy as np
import pytest
import torch

from oracle import oracle_np as O
from paper_2603_02402_b200 import synth
import parity_util as U
from paper_2603_02402_b200 import binding as B  # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2603_02402_b200 import build, binding
    build.build()
    binding.lib()
    assert torch.cuda.is_available()


SMALL = [  # n, G, seed, depth, empty_rows, empty_genes  (several tiles + ragged tails + empties)
    (1, 1, 0, 3.0, (), ()),
    (3, 7, 1, 2.0, (1,), (2,)),
    (257, 1031, 2, 0.7, (0, 100, 256), (0, 1030)),
    (1500, 4099, 3, 0.4, (17,), (5, 6, 7)),
    (700, 18000, 4, 0.158, (), ()),
    (33, 36000, 5, 0.6, (32,), ()),
]


def _flags(G, seed):
    rng = np.random.default_rng(1000 + seed)
    f = (rng.random(G) < 0.05).astype(np.uint8)
    f[: min(13, G)] = 1
    return f


def _shuffle_rows_cols(indptr, indices, data, seed):
    """Same matrix with the entries of every row in random column order (unsorted CSR)."""
    rng = np.random.default_rng(seed)
    idx2, dat2 = indices.copy(), data.copy()
    for i in range(len(indptr) - 1):
        lo, hi = indptr[i], indptr[i + 1]
        p = rng.permutation(hi - lo)
        idx2[lo:hi] = indices[lo:hi][p]; dat2[lo:hi] = data[lo:hi][p]
    return idx2, dat2


@pytest.mark.parametrize("n,G,seed,depth,er,eg", SMALL)
@pytest.mark.parametrize("sorted_rows", [True, False])
def test_qc_metrics(n, G, seed, depth, er, eg, sorted_rows):
    from paper_2603_02402_b200 import rsc_qc_metrics
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    if not sorted_rows:
        indices, data = _shuffle_rows_cols(indptr, indices, data, seed)
    flags = _flags(G, seed)
    want = O.qc_metrics(indptr, indices, data, G, flags)
    X = U.to_dev(indptr, indices, data, G, sorted_rows)
    got = rsc_qc_metrics(X, torch.as_tensor(flags).cuda())
    torch.cuda.synchronize()
    for k in ("cell_total_i64", "cell_n_genes", "cell_flag_total_i64", "gene_n_cells", "gene_total_i64"):
        U.assert_int_equal(got[k], want[k], k)
    U.assert_f32_close(got["cell_total_f32"], want["cell_total_f32"], "cell_total_f32", rtol=0)
    U.assert_f32_close(got["cell_flag_pct"], want["cell_flag_pct"], "cell_flag_pct")
    # invariants
    assert int(got["gene_n_cells"].sum()) == int(got["cell_n_genes"].sum()) == len(indices)
    assert int(got["gene_total_i64"].sum()) == int(got["cell_total_i64"].sum())
    # no flags -> zero flagged totals
    got0 = rsc_qc_metrics(X, None)
    assert int(got0["cell_flag_total_i64"].abs().sum()) == 0


@pytest.mark.parametrize("n,G,seed,depth,er,eg", SMALL)
@pytest.mark.parametrize("s", [1e4, 1e6])
def test_normalize_then_log1p(n, G, seed, depth, er, eg, s):
    from paper_2603_02402_b200 import rsc_normalize_total, rsc_log1p, rsc_qc_metrics
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    xn_o, scale_o = O.normalize_total(indptr, data, s)
    xl_o = O.log1p(xn_o)
    X = U.to_dev(indptr, indices, data, G)
    scale = rsc_normalize_total(X, s, None, return_scale=True)
    U.assert_f32_close(X.data, xn_o, "x' (totals summed by the kernel)")
    U.assert_f32_close(scale, scale_o.astype(np.float32), "scale")
    # with the exact int64 totals from QC: bit-identical to the self-summed variant
    X2 = U.to_dev(indptr, indices, data, G)
    q = rsc_qc_metrics(X2)
    rsc_normalize_total(X2, s, q["cell_total_i64"])
    assert torch.equal(X.data, X2.data)
    # invariant: row sums equal target_sum
    rows = np.repeat(np.arange(n), np.diff(indptr))
    rs = np.bincount(rows, weights=U.np_(X.data).astype(np.float64), minlength=n)
    ne = np.diff(indptr) > 0
    assert np.all(np.abs(rs[ne] - s) <= s * 1e-6)
    rsc_log1p(X)
    U.assert_f32_close(X.data, xl_o, "x''")
    assert torch.equal(X.indices.cpu(), torch.as_tensor(indices))       # pattern untouched
    assert np.all((U.np_(X.data) == 0) == (xn_o == 0))


def test_log1p_value_range_and_alignment():
    """Tiny / huge / zero arguments and every 16-byte misalignment of the data pointer."""
    from paper_2603_02402_b200 import rsc_log1p, Csr
    vals = np.concatenate([[0.0, 1e-30, 1e-10, 1e-7, 1e-5, 1e-3, 0.02, 0.03, 0.0312, 0.0313, 0.1, 0.5,
                            1.0, np.e - 1, 10, 1e4, 1e6, 3e7, 1e20],
                           np.exp(np.random.default_rng(0).uniform(-20, 20, 5000))]).astype(np.float32)
    want = O.log1p(vals)
    for off in range(4):
        for length in (len(vals), 1, 2, 3, 5, 8, 1023):
            base = torch.zeros(len(vals) + 8, dtype=torch.float32, device="cuda")
            view = base[off:off + length]
            view.copy_(torch.as_tensor(vals[:length]))
            X = Csr(torch.tensor([0, length], dtype=torch.int64, device="cuda"),
                    torch.zeros(length, dtype=torch.int32, device="cuda"), view, 1)
            rsc_log1p(X)
            U.assert_f32_close(view, want[:length], f"log1p off={off} len={length}")
            assert float(base[:off].abs().sum()) == 0 and float(base[off + length:].abs().sum()) == 0


@pytest.mark.parametrize("n,G,seed,depth,er,eg", SMALL[1:])
@pytest.mark.parametrize("sorted_rows", [True, False])
def test_gene_moments(n, G, seed, depth, er, eg, sorted_rows):
    from paper_2603_02402_b200 import rsc_gene_moments
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    xl = O.log1p(O.normalize_total(indptr, data, 1e4)[0])
    if not sorted_rows:
        indices, xl = _shuffle_rows_cols(indptr, indices, xl, seed)
    X = U.to_dev(indptr, indices, xl, G, sorted_rows)
    for transform in (0, 1):
        for ddof in (1, 0):
            mo, vo, s1o, s2o = O.gene_moments(indptr, indices, xl, G, transform, ddof)
            g = rsc_gene_moments(X, transform, ddof)
            U.assert_moments_close(g["mean"], g["var"], mo, vo, f"moments t={transform} ddof={ddof}")
            np.testing.assert_allclose(U.np_(g["sum"]), s1o, rtol=1e-12)
            # S2 of the three-word integer scheme is a sum of squares each rounded to <= 2^-39
            # of the smallest representable square (2^-39); the bar is 1e-9
            np.testing.assert_allclose(U.np_(g["sumsq"]), s2o, rtol=4e-12)
    assert torch.equal(X.data.cpu(), torch.as_tensor(xl))               # read-only


@pytest.mark.parametrize("n,G,seed,depth,er,eg", SMALL[1:])
@pytest.mark.parametrize("s", [1e4, 1e6])
@pytest.mark.parametrize("which", [1, 2, 3])
@pytest.mark.parametrize("sorted_rows", [True, False])
def test_fused_normalize_log1p_moments(n, G, seed, depth, er, eg, s, which, sorted_rows):
    from paper_2603_02402_b200 import (rsc_normalize_log1p_moments, rsc_normalize_total,
                                       rsc_qc_metrics)
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    if not sorted_rows:
        indices, data = _shuffle_rows_cols(indptr, indices, data, seed)
    X = U.to_dev(indptr, indices, data, G, sorted_rows)
    Xn = U.clone(X)
    q = rsc_qc_metrics(X)
    out = rsc_normalize_log1p_moments(X, s, q["cell_total_i64"], q["gene_n_cells"], which, 1)
    # (a) values against the independent oracle chain
    xl_o = O.log1p(O.normalize_total(indptr, data, s)[0])
    U.assert_f32_close(X.data, xl_o, "fused x''")
    # (b) log-scale moments: oracle M1 on the very x'' the kernel wrote (bit-identical input)
    if which & 1:
        mo, vo, _, _ = O.gene_moments(indptr, indices, U.np_(X.data), G, 0, 1)
        U.assert_moments_close(out["mean_log"], out["var_log"], mo, vo, "fused log moments")
    # (c) linear-scale moments: oracle M1 on x' written by rsc_normalize_total (same fp32 expr)
    if which & 2:
        rsc_normalize_total(Xn, s, q["cell_total_i64"])
        mo, vo, _, _ = O.gene_moments(indptr, indices, U.np_(Xn.data), G, 0, 1)
        U.assert_moments_close(out["mean_lin"], out["var_lin"], mo, vo, "fused lin moments")
    # (d) independent chains end to end at 1e-6
    if which & 1:
        mo, vo, _, _ = O.gene_moments(indptr, indices, xl_o, G, 0, 1)
        np.testing.assert_allclose(U.np_(out["mean_log"]), mo, rtol=1e-6, atol=1e-300)
        np.testing.assert_allclose(U.np_(out["var_log"]), vo, rtol=1e-6, atol=1e-12)


@pytest.mark.parametrize("G,seed,n_top,n_bins", [(1, 0, 1, 20), (2, 1, 1, 20), (50, 2, 5, 20),
                                                 (1000, 3, 100, 20), (4099, 4, 500, 7),
                                                 (18000, 5, 2000, 20), (36000, 6, 3000, 20),
                                                 (30000, 7, 40000, 20), (5000, 8, 1, 1)])
@pytest.mark.parametrize("log_flag", [1, 0])
def test_hvg_select_same_inputs(G, seed, n_top, n_bins, log_flag):
    from paper_2603_02402_b200 import rsc_hvg_select
    rng = np.random.default_rng(seed)
    mean = np.exp(rng.normal(-3, 2, G))
    var = mean * np.exp(rng.normal(0.2, 0.6, G))
    dead = rng.random(G) < 0.1
    mean[dead] = 0.0; var[dead] = 0.0                      # undetected genes
    if G > 10:
        var[3] = 0.0                                       # zero dispersion -> NaN under the log
        mean[7] = mean[8]; var[7] = var[8]                 # exact tie
    o = O.hvg_select(mean, var, n_top, n_bins, seurat_log=bool(log_flag))
    g = rsc_hvg_select(torch.as_tensor(mean).cuda(), torch.as_tensor(var).cuda(), n_top, n_bins, log_flag)
    torch.cuda.synchronize()
    U.assert_hvg_matches(g, o, n_top, f"hvg G={G}", strict=False)


def test_hvg_many_ties_takes_the_general_selection_path():
    """5000 genes in one bin with only two distinct dispersions: 2500 equal z-scores sit in
    the value bin that holds the cutoff -- more than the fast top-k path gathers -- so the
    8-pass radix select runs; every tie at the cutoff is selected (reading R13 / H7)."""
    from paper_2603_02402_b200 import rsc_hvg_select
    G = 5000
    mean = 1.0 + np.arange(G) / 8192.0                    # dyadic: var / mean is exactly 3 or 0.5
    var = mean * np.where(np.arange(G) % 2 == 0, 3.0, 0.5)
    for n_bins, log_flag in ((1, 1), (1, 0)):
        o = O.hvg_select(mean, var, 100, n_bins, seurat_log=bool(log_flag))
        g = rsc_hvg_select(torch.as_tensor(mean).cuda(), torch.as_tensor(var).cuda(), 100, n_bins, log_flag)
        torch.cuda.synchronize()
        U.assert_hvg_matches(g, o, 100, f"ties n_bins={n_bins} log={log_flag}", strict=False)
        assert int(U.np_(g["count"])[0]) == int(o["mask"].sum()) == G // 2


def test_hvg_golden_and_degenerate():
    from paper_2603_02402_b200 import rsc_hvg_select
    # hand-worked fixture (tests/golden/hvg_tiny.txt, case two_bins / single_gene_bin_and_tie)
    mean = torch.tensor([1, 2, 3, 4, 5, 6, 7, 8], dtype=torch.float64).cuda()
    var = torch.tensor([1, 6, 15, 28, 10, 12, 14, 80], dtype=torch.float64).cuda()
    g = rsc_hvg_select(mean, var, 3, 2, 0)
    assert U.np_(g["indices"])[:3].tolist() == [2, 3, 7] and int(g["count"][0]) == 3
    assert U.np_(g["bin"]).tolist() == [0, 0, 0, 0, 1, 1, 1, 1]
    np.testing.assert_allclose(U.np_(g["disp_norm"])[4:], [-0.5, -0.5, -0.5, 1.5], rtol=1e-14)
    mean = torch.tensor([1, 2, 3, 10], dtype=torch.float64).cuda()
    var = torch.tensor([2, 8, 18, 50], dtype=torch.float64).cuda()
    g = rsc_hvg_select(mean, var, 1, 3, 0)
    assert int(g["count"][0]) == 2 and U.np_(g["indices"])[:2].tolist() == [2, 3]   # tie at cutoff
    assert U.np_(g["disp_norm"]).tolist() == [-1.0, 0.0, 1.0, 1.0]
    # all means equal (reading R10): one bin, still a valid selection
    mean = np.full(64, 2.5); var = np.linspace(1, 5, 64)
    o = O.hvg_select(mean, var, 8, 20)
    g = rsc_hvg_select(torch.as_tensor(mean).cuda(), torch.as_tensor(var).cuda(), 8, 20, 1)
    U.assert_hvg_matches(g, o, 8, "degenerate")
    # nothing valid -> empty selection
    z = torch.zeros(16, dtype=torch.float64).cuda()
    g = rsc_hvg_select(z, z, 4, 20, 1)
    assert int(g["count"][0]) == 0 and int(g["mask"].sum()) == 0


def test_errors_are_loud():
    from paper_2603_02402_b200 import binding as B
    indptr, indices, data, _ = synth.small_nb_csr(10, 20, 0, 1.0)
    X = U.to_dev(indptr, indices, data, 20)
    with pytest.raises(B.RscError):
        B.rsc_normalize_total(X, float("nan"))
    with pytest.raises(B.RscError):
        B.rsc_gene_moments(X, transform=2)
    with pytest.raises(B.RscError):
        B.rsc_hvg_select(torch.zeros(4, dtype=torch.float64).cuda(), torch.zeros(4, dtype=torch.float64).cuda(), 0)
    # too-small workspace is refused
    import ctypes as C
    L = B.lib()
    cs = X.c_struct()
    m = torch.empty(20, dtype=torch.float64, device="cuda")
    rc = L.rsc_gene_moments(C.byref(cs), 0, 1, B._ptr(m), B._ptr(m), None, None, B._ptr(m), 8, None)
    assert rc == B.RSC_ERR_WORKSPACE


# ----------------------------------------------------------------------------------------
# streaming kernels: row split table, flush paths, accumulator modes
# ----------------------------------------------------------------------------------------
def _splits_ref(indptr, indices, G, width=1024):
    """splits[row, k] = #{entries of the row with column < k * width} (definition in rsc.h)."""
    K = (G + width - 1) // width
    n = len(indptr) - 1
    out = np.zeros((n, K + 1), dtype=np.int64)
    for i in range(n):
        cols = indices[indptr[i]:indptr[i + 1]]
        for k in range(K + 1):
            out[i, k] = int(np.sum(cols < k * width))
    return out


@pytest.mark.parametrize("n,G,seed,depth,er,eg", SMALL)
def test_row_splits_qc_and_standalone(n, G, seed, depth, er, eg):
    from paper_2603_02402_b200 import binding as B
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    want = _splits_ref(indptr, indices, G)
    X = U.to_dev(indptr, indices, data, G)
    assert B.rsc_row_splits_count(n, G) == want.size
    a = U.np_(B.rsc_row_splits(X)).astype(np.int64)[: want.size].reshape(want.shape)
    q = B.rsc_qc_metrics(X, None, with_row_splits=True)
    b = U.np_(q["row_splits"]).astype(np.int64)[: want.size].reshape(want.shape)
    assert np.array_equal(a, want), "rsc_row_splits"
    assert np.array_equal(b, want), "row splits emitted by rsc_qc_metrics"
    # only the entries the fused pass reads (rsc_qc_metrics_splits): the listed columns of the
    # table are exact, and the fused pass fed with that partial table gives the same moments
    for which in (1, 3):
        need = B.rsc_moments_split_blocks(G, which)
        K = want.shape[1] - 1
        assert need and need[0] == 0 and need[-1] == K and need == sorted(set(need))
        qp = B.rsc_qc_metrics(X, None, with_row_splits=True, split_blocks=need)
        c = U.np_(qp["row_splits"]).astype(np.int64)[: want.size].reshape(want.shape)
        assert np.array_equal(c[:, need], want[:, need]), "partial row split table"
        X1, X2 = U.clone(X), U.clone(X)
        o1 = B.rsc_normalize_log1p_moments(X1, 1e4, q["cell_total_i64"], q["gene_n_cells"], which, 0,
                                           row_splits=q["row_splits"], return_sums=True)
        o2 = B.rsc_normalize_log1p_moments(X2, 1e4, q["cell_total_i64"], q["gene_n_cells"], which, 0,
                                           row_splits=qp["row_splits"], return_sums=True)
        assert torch.equal(X1.data, X2.data)
        np.testing.assert_allclose(U.np_(o1["sums"]), U.np_(o2["sums"]), rtol=1e-14)


@pytest.fixture
def small_budgets():
    """Force many flushes of the CTA-private tables and a small grid (rsc_set_option)."""
    from paper_2603_02402_b200 import binding as B
    B.rsc_set_option("fused_row_budget", 8)
    B.rsc_set_option("flush_all", 1)
    B.rsc_set_option("qc_row_budget", 8)
    B.rsc_set_option("grid_ctas", 9)
    yield
    B.rsc_set_option("fused_row_budget", 256)
    B.rsc_set_option("flush_all", 0)
    B.rsc_set_option("qc_row_budget", 512)
    B.rsc_set_option("grid_ctas", 0)


@pytest.mark.parametrize("n,G,seed,depth,er,eg", SMALL[2:])
@pytest.mark.parametrize("which", [1, 2, 3, 7])
def test_streaming_kernels_flush_paths(small_budgets, n, G, seed, depth, er, eg, which):
    from paper_2603_02402_b200 import binding as B
    indptr, indices, data, _ = synth.small_nb_csr(n, G, seed, depth, empty_rows=er, empty_genes=eg)
    flags = _flags(G, seed)
    want = O.qc_metrics(indptr, indices, data, G, flags)
    X = U.to_dev(indptr, indices, data, G)
    Xn = U.clone(X)
    q = B.rsc_qc_metrics(X, torch.as_tensor(flags).cuda(), with_row_splits=True)
    for k in ("cell_total_i64", "cell_n_genes", "cell_flag_total_i64", "gene_n_cells", "gene_total_i64"):
        U.assert_int_equal(q[k], want[k], k)
    s = 1e4
    out = B.rsc_normalize_log1p_moments(X, s, q["cell_total_i64"], q["gene_n_cells"], which, 1,
                                        row_splits=q["row_splits"])
    xl_o = O.log1p(O.normalize_total(indptr, data, s)[0])
    U.assert_f32_close(X.data, xl_o, "x''")
    if which & 1:
        mo, vo, _, _ = O.gene_moments(indptr, indices, U.np_(X.data), G, 0, 1)
        U.assert_moments_close(out["mean_log"], out["var_log"], mo, vo, "log moments")
    if which & 2:
        B.rsc_normalize_total(Xn, s, q["cell_total_i64"])
        mo, vo, _, _ = O.gene_moments(indptr, indices, U.np_(Xn.data), G, 0, 1)
        U.assert_moments_close(out["mean_lin"], out["var_lin"], mo, vo, "lin moments")


def test_fused_equals_unfused_bitwise_and_is_order_independent():
    """The fused pass writes the very x'' that rsc_normalize_total + rsc_log1p write, and its
    integer sums (on chip and in global memory) do not depend on the order of the atomic adds, the
    CTA schedule or the grid: the moments are bit-reproducible."""
    from paper_2603_02402_b200 import binding as B
    indptr, indices, data, _ = synth.small_nb_csr(1500, 4099, 3, 0.4)
    X = U.to_dev(indptr, indices, data, 4099)
    Xu = U.clone(X)
    q = B.rsc_qc_metrics(X)
    out1 = B.rsc_normalize_log1p_moments(X, 1e4, q["cell_total_i64"], q["gene_n_cells"], 3, 1, return_sums=True)
    B.rsc_normalize_total(Xu, 1e4, q["cell_total_i64"])
    B.rsc_log1p(Xu)
    assert torch.equal(X.data, Xu.data)
    X2 = U.to_dev(indptr, indices, data, 4099)
    B.rsc_set_option("grid_ctas", 37)
    try:
        out2 = B.rsc_normalize_log1p_moments(X2, 1e4, q["cell_total_i64"], None, 3, 1, return_sums=True)
    finally:
        B.rsc_set_option("grid_ctas", 0)
    # on-chip sums and the global totals are integers: the sums do not depend on the grid, the
    # CTA schedule or the order of the atomic adds -- bit-identical
    assert np.array_equal(U.np_(out1["sums"]), U.np_(out2["sums"]))
    X3 = U.to_dev(indptr, indices, data, 4099)
    out3 = B.rsc_normalize_log1p_moments(X3, 1e4, q["cell_total_i64"], q["gene_n_cells"], 3, 1, return_sums=True)
    assert np.array_equal(U.np_(out1["sums"]), U.np_(out3["sums"]))
    for k in ("mean_log", "var_log", "mean_lin", "var_lin"):
        assert torch.equal(out1[k], out2[k]) and torch.equal(out1[k], out3[k]), k


def test_fixed_point_extreme_ranges():
    """Rows whose totals differ by 2^26 (x' from ~1e-4 to target_sum) and both target sums: the
    integer accumulators are exact inside their window (one-word and two-word addends), and the
    values below it (the deep cell's) take the global double path."""
    from paper_2603_02402_b200 import binding as B
    rng = np.random.default_rng(7)
    n, G = 64, 3000
    dense = np.zeros((n, G), dtype=np.float64)
    for i in range(n):
        k = rng.integers(1, 40)
        cols = rng.choice(G, size=k, replace=False)
        dense[i, cols] = rng.integers(1, 4, size=k)
    dense[0, :] = 0; dense[0, 5] = 7                      # one gene takes the whole cell: x' = s
    dense[1, :2000] = 500.0                               # T = 1e6: x' = s / 2000 * ... tiny
    dense[2, 5] = 1.0; dense[2, 100:1100] = 1000.0        # x' of gene 5 ~ s * 1e-6
    dense[3, :] = 0; dense[3, 10:74] = 1.0e6; dense[3, 5] = 3.0   # T = 6.4e7: x' below any window
    indptr = np.zeros(n + 1, dtype=np.int64)
    r, c = np.nonzero(dense)
    np.cumsum(np.bincount(r, minlength=n), out=indptr[1:])
    indices = c.astype(np.int32); data = dense[r, c].astype(np.float32)
    for s in (1e4, 1e6):
        for which in (3, 7):
            X = U.to_dev(indptr, indices, data, G)
            Xn = U.clone(X)
            q = B.rsc_qc_metrics(X)
            out = B.rsc_normalize_log1p_moments(X, s, q["cell_total_i64"], q["gene_n_cells"], which, 1)
            mo, vo, _, _ = O.gene_moments(indptr, indices, U.np_(X.data), G, 0, 1)
            U.assert_moments_close(out["mean_log"], out["var_log"], mo, vo, f"log s={s} which={which}")
            B.rsc_normalize_total(Xn, s, q["cell_total_i64"])
            mo, vo, _, _ = O.gene_moments(indptr, indices, U.np_(Xn.data), G, 0, 1)
            U.assert_moments_close(out["mean_lin"], out["var_lin"], mo, vo, f"lin s={s} which={which}")


def test_edge_inputs_misaligned_explicit_zeros_and_empty():
    """(a) indices / data at every 4-byte misalignment of the 16-byte quads (served by the generic
    kernels): same results as the aligned streaming kernels; (b) explicit stored zeros are not
    "detected" (reading R2) and stay zero through log1p; (c) a matrix of empty rows."""
    from paper_2603_02402_b200 import binding as B, Csr
    n, G, s = 300, 2100, 1e4
    indptr, indices, data, _ = synth.small_nb_csr(n, G, 11, 0.5, empty_rows=(0, 299), empty_genes=(7,))
    data = data.copy()
    data[::17] = 0.0                                       # explicit zeros
    flags = _flags(G, 11)
    q_o = O.qc_metrics(indptr, indices, data, G, flags)
    assert q_o["cell_n_genes"].sum() < len(data)           # the zeros are stored but not counted
    ref = None
    for off in range(4):
        ib = torch.zeros(len(indices) + 8, dtype=torch.int32, device="cuda")
        db = torch.zeros(len(data) + 8, dtype=torch.float32, device="cuda")
        iv, dv = ib[off:off + len(indices)], db[off:off + len(data)]
        iv.copy_(torch.as_tensor(indices)); dv.copy_(torch.as_tensor(data))
        X = Csr(torch.as_tensor(indptr).cuda(), iv, dv, G)
        q = B.rsc_qc_metrics(X, torch.as_tensor(flags).cuda())
        for k in ("cell_total_i64", "cell_n_genes", "cell_flag_total_i64", "gene_n_cells", "gene_total_i64"):
            U.assert_int_equal(q[k], q_o[k], f"{k} off={off}")
        out = B.rsc_normalize_log1p_moments(X, s, q["cell_total_i64"], q["gene_n_cells"], 3, 1)
        xl = U.np_(X.data)
        assert np.all((xl == 0) == (data == 0))
        mo, vo, _, _ = O.gene_moments(indptr, indices, xl, G, 0, 1)
        U.assert_moments_close(out["mean_log"], out["var_log"], mo, vo, f"log off={off}")
        if ref is None:
            ref = xl.copy()
        else:
            assert np.array_equal(xl, ref), "aligned and misaligned paths write different x''"
        assert float(db[:off].abs().sum()) == 0 and float(db[off + len(data):].abs().sum()) == 0
    # (c) only empty rows
    X = Csr(torch.zeros(6, dtype=torch.int64, device="cuda"), torch.zeros(0, dtype=torch.int32, device="cuda"),
            torch.zeros(0, dtype=torch.float32, device="cuda"), 50)
    q = B.rsc_qc_metrics(X)
    assert int(q["cell_total_i64"].abs().sum()) == 0 and int(q["gene_n_cells"].abs().sum()) == 0
    out = B.rsc_normalize_log1p_moments(X, s, q["cell_total_i64"], q["gene_n_cells"], 3, 1)
    assert float(out["mean_log"].abs().sum()) == 0 and float(out["var_lin"].abs().sum()) == 0


@pytest.mark.parametrize("G,n_top,n_bins", [(7, 3, 20), (1000, 100, 20), (18000, 2000, 20), (36000, 3000, 32), (65536, 5000, 7)])
def test_hvg_cluster_kernel_equals_single_cta(G, n_top, n_bins):
    """The cluster kernel (default) and the one-CTA kernel give the same bins, mask, indices and
    count, and z-scores that differ only by the summation order inside a bin."""
    rng = np.random.default_rng(G)
    mean = np.exp(rng.normal(-1.0, 1.5, G)); var = mean * np.exp(rng.normal(0.3, 0.6, G))
    mean[rng.choice(G, max(1, G // 50), replace=False)] = 0.0
    var[mean == 0] = 0.0
    gm, gv = torch.from_numpy(mean).cuda(), torch.from_numpy(var).cuda()
    a = B.rsc_hvg_select(gm, gv, n_top, n_bins)
    B.rsc_set_option("hvg_single_cta", 1)
    try:
        b = B.rsc_hvg_select(gm, gv, n_top, n_bins)
    finally:
        B.rsc_set_option("hvg_single_cta", 0)
    torch.cuda.synchronize()
    assert torch.equal(a["bin"], b["bin"]) and torch.equal(a["mean_t"], b["mean_t"])
    assert torch.equal(torch.nan_to_num(a["disp"], nan=-9.0), torch.nan_to_num(b["disp"], nan=-9.0))
    za, zb = a["disp_norm"].cpu().numpy(), b["disp_norm"].cpu().numpy()
    np.testing.assert_allclose(za, zb, rtol=1e-11, atol=1e-12, equal_nan=True)
    ca, cb = int(a["count"][0]), int(b["count"][0])
    ma, mb = a["mask"].cpu().numpy().astype(bool), b["mask"].cpu().numpy().astype(bool)
    d = np.nonzero(ma != mb)[0]                       # only z values tied within rounding at the cutoff may differ
    if len(d):
        cut = np.sort(zb[~np.isnan(zb)])[::-1][min(n_top, (~np.isnan(zb)).sum()) - 1]
        assert np.all(np.abs(zb[d] - cut) <= 1e-9 * max(1.0, abs(cut)))
    assert np.array_equal(a["indices"].cpu().numpy()[:ca], np.nonzero(ma)[0]) and ca == ma.sum() and cb == mb.sum()
    o = O.hvg_select(mean, var, n_top, n_bins)
    U.assert_hvg_matches(a, o, n_top, f"cluster G={G}", strict=False)


@pytest.mark.parametrize("case", ["one_bin", "all_equal_means", "infinite_z", "all_nan", "n_top_huge", "max_bins"])
def test_hvg_cluster_kernel_degenerate_cases(case):
    """Degenerate inputs through the cluster kernel against the oracle (and the one-CTA kernel)."""
    rng = np.random.default_rng(5)
    G, n_top, n_bins = 3000, 300, 20
    mean = np.exp(rng.normal(-1.0, 1.5, G)); var = mean * np.exp(rng.normal(0.3, 0.6, G))
    if case == "one_bin":
        n_bins = 1
    elif case == "all_equal_means":
        mean[:] = 0.7
    elif case == "infinite_z":                       # a bin whose members share one dispersion: sd = 0 -> z = 0/0 or x/0
        mean[:40] = np.linspace(5.0, 5.001, 40); var[:40] = 2.0 * mean[:40]
        mean[40] = 5.0005; var[40] = 9.0 * mean[40]
        n_bins = 32
    elif case == "all_nan":
        var[:] = 0.0                                 # d = 0 -> NaN after the Seurat transform: nothing is selectable
    elif case == "n_top_huge":
        n_top = 10 * G
    elif case == "max_bins":
        n_bins = 32
    gm, gv = torch.from_numpy(mean).cuda(), torch.from_numpy(var).cuda()
    a = B.rsc_hvg_select(gm, gv, n_top, n_bins)
    B.rsc_set_option("hvg_single_cta", 1)
    try:
        b = B.rsc_hvg_select(gm, gv, n_top, n_bins)
    finally:
        B.rsc_set_option("hvg_single_cta", 0)
    torch.cuda.synchronize()
    o = O.hvg_select(mean, var, n_top, n_bins)
    U.assert_hvg_matches(a, o, n_top, f"cluster {case}", strict=False)
    U.assert_hvg_matches(b, o, n_top, f"one CTA {case}", strict=False)
    assert torch.equal(a["bin"], b["bin"]) and int(a["count"][0]) == int(b["count"][0])
    assert torch.equal(a["mask"], b["mask"])
