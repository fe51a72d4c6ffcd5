"""Pins for the oracle's gene moments (M1) and HVG selection (H1..H7).

Expected values come from numpy / pandas library routines on dense data,
closed forms, invariants, explicit loops and a hand-worked fixture — never
from the oracle itself.
"""
import os

import numpy as np
import pandas as pd
import pytest

from oracle import oracle_np as O
from paper_2603_02402_b200 import synth

HERE = os.path.dirname(os.path.abspath(__file__))

CASES = [(1, 3, 0, 3.0), (2, 4, 1, 2.0), (40, 33, 2, 1.0), (64, 200, 3, 0.5), (130, 97, 4, 1.5)]


def _dense(indptr, indices, vals, n, G):
    D = np.zeros((n, G))
    rows = np.repeat(np.arange(n), np.diff(indptr))
    D[rows, indices] = vals
    return D


@pytest.mark.parametrize("n,G,seed,depth", CASES)
@pytest.mark.parametrize("ddof", [0, 1])
def test_moments_vs_numpy_dense(n, G, seed, depth, ddof):
    if n - ddof <= 0:
        pytest.skip("variance undefined")
    indptr, indices, data, X = synth.small_nb_csr(n, G, seed, depth, empty_genes=(1,))
    xl = O.log1p(O.normalize_total(indptr, data, 1e4)[0])
    mean, var, s1, s2 = O.gene_moments(indptr, indices, xl, G, 0, ddof)
    D = _dense(indptr, indices, xl.astype(np.float64), n, G)
    np.testing.assert_allclose(mean, D.mean(axis=0), rtol=1e-13, atol=0)
    np.testing.assert_allclose(var, D.var(axis=0, ddof=ddof), rtol=1e-11, atol=1e-300)
    np.testing.assert_allclose(s1, D.sum(axis=0), rtol=1e-13)
    np.testing.assert_allclose(s2, (D * D).sum(axis=0), rtol=1e-13)
    assert mean[1] == 0 and var[1] == 0          # all-zero gene
    # transform = expm1 un-logs first (reading R8)
    mean_e, var_e, _, _ = O.gene_moments(indptr, indices, xl, G, 1, ddof)
    E = np.expm1(D)
    np.testing.assert_allclose(mean_e, E.mean(axis=0), rtol=1e-13)
    np.testing.assert_allclose(var_e, E.var(axis=0, ddof=ddof), rtol=1e-11, atol=1e-300)


def test_moments_closed_forms():
    n, G = 10, 4
    # gene 0: constant 2.5 in every cell -> mean 2.5 var 0
    # gene 1: single entry v=3 -> mean v/n, var(ddof=1) = v^2/n
    # gene 2: values 1..10 -> mean 5.5, var 55/6 ; gene 3: empty
    rows, cols, vals = [], [], []
    for i in range(n):
        rows += [i, i]; cols += [0, 2]; vals += [2.5, float(i + 1)]
    rows.append(4); cols.append(1); vals.append(3.0)
    order = np.lexsort((cols, rows))
    rows = np.array(rows)[order]; cols = np.array(cols, np.int32)[order]; vals = np.array(vals, np.float32)[order]
    indptr = np.zeros(n + 1, np.int64); np.cumsum(np.bincount(rows, minlength=n), out=indptr[1:])
    mean, var, s1, s2 = O.gene_moments(indptr, cols, vals, G, 0, 1)
    assert mean[0] == 2.5 and var[0] == 0.0
    assert mean[1] == 0.3 and abs(var[1] - 0.9) < 1e-15
    assert mean[2] == 5.5 and abs(var[2] - 55.0 / 6.0) < 1e-14
    assert mean[3] == 0 and var[3] == 0
    _, var0, _, _ = O.gene_moments(indptr, cols, vals, G, 0, 0)
    np.testing.assert_allclose(var0 * n / (n - 1), var, rtol=1e-15)   # ddof ratio n/(n-1)


def test_moments_permutation_invariance():
    indptr, indices, data, X = synth.small_nb_csr(50, 30, 7, 1.0)
    m0, v0, _, _ = O.gene_moments(indptr, indices, data, 30)
    perm = np.random.default_rng(0).permutation(50)
    Xp = X[perm]
    nzr, nzc = np.nonzero(Xp)
    ip = np.zeros(51, np.int64); np.cumsum(np.bincount(nzr, minlength=50), out=ip[1:])
    m1, v1, _, _ = O.gene_moments(ip, nzc.astype(np.int32), Xp[nzr, nzc].astype(np.float32), 30)
    np.testing.assert_allclose(m0, m1, rtol=1e-14); np.testing.assert_allclose(v0, v1, rtol=1e-12)


# ------------------------------------------------------------------ HVG
@pytest.mark.parametrize("seed", range(40))
@pytest.mark.parametrize("n_bins", [20, 7])
def test_bins_match_pandas_cut(seed, n_bins):
    rng = np.random.default_rng(seed)
    G = int(rng.integers(2, 400))
    m = np.log1p(np.exp(rng.normal(-2, 2, G)))
    if seed % 5 == 0:
        m[rng.integers(0, G, 3)] = m.max()       # repeated extreme values
    edges = O.bin_edges(m, n_bins)
    codes = O.assign_bins(m, edges)
    cat, pbins = pd.cut(m, bins=n_bins, retbins=True)
    assert np.array_equal(edges, pbins)                          # bit-identical edges
    assert np.array_equal(codes, np.asarray(cat.codes))


def test_bins_degenerate_matches_pandas_cut():
    for val in (0.0, 2.5, 1e-12):
        m = np.full(9, val)
        edges = O.bin_edges(m, 20)
        cat, pbins = pd.cut(m, bins=20, retbins=True)
        assert np.array_equal(edges, pbins)
        assert np.array_equal(O.assign_bins(m, edges), np.asarray(cat.codes))


def _hvg_bruteforce(mean, var, n_top, n_bins):
    """Independent restatement using pandas cut / groupby (skipna mean, std ddof=1)."""
    mean = np.array(mean, float); var = np.array(var, float)
    mean[mean == 0] = 1e-12
    with np.errstate(all="ignore"):
        d = var / mean
        d[d == 0] = np.nan
        d = np.log(d); m = np.log1p(mean)
    df = pd.DataFrame({"m": m, "d": d})
    df["bin"] = pd.cut(df["m"], bins=n_bins)
    grp = df.groupby("bin", observed=False)["d"]
    mu = grp.mean(); sd = grp.std(ddof=1); cnt = grp.count()
    one = cnt == 1
    sd[one] = mu[one]; mu[one] = 0.0
    z = (df["d"].values - mu[df["bin"]].values.astype(float)) / sd[df["bin"]].values.astype(float)
    valid = ~np.isnan(z)
    k = min(n_top, int(valid.sum()))
    order = np.argsort(-np.where(valid, z, -np.inf), kind="stable")
    cutoff = z[order[k - 1]] if k > 0 else np.nan
    mask = valid & (z >= cutoff)
    return d, m, z, mask


@pytest.mark.parametrize("n,G,seed,depth", [(60, 300, 11, 0.6), (200, 1000, 12, 0.3), (30, 40, 13, 2.0)])
@pytest.mark.parametrize("which", ["lin", "log"])
def test_hvg_vs_pandas_bruteforce(n, G, seed, depth, which):
    indptr, indices, data, X = synth.small_nb_csr(n, G, seed, depth, empty_genes=(0, 5))
    xn = O.normalize_total(indptr, data, 1e4)[0]
    v = xn if which == "lin" else O.log1p(xn)
    mean, var, _, _ = O.gene_moments(indptr, indices, v, G)
    n_top = max(1, G // 10)
    h = O.hvg_select(mean, var, n_top, 20)
    d, m, z, mask = _hvg_bruteforce(mean, var, n_top, 20)
    np.testing.assert_array_equal(np.isnan(h["disp"]), np.isnan(d))
    np.testing.assert_allclose(h["disp"], d, rtol=1e-14, equal_nan=True)
    np.testing.assert_allclose(h["mean_t"], m, rtol=1e-15)
    np.testing.assert_allclose(h["disp_norm"], z, rtol=1e-10, atol=1e-12, equal_nan=True)
    assert np.array_equal(h["mask"].astype(bool), mask)
    assert h["count"] == mask.sum() >= min(n_top, (~np.isnan(z)).sum())
    assert np.array_equal(h["indices"], np.nonzero(mask)[0])
    # all-zero genes: NaN dispersion, never selected
    assert np.isnan(h["disp_norm"][0]) and h["mask"][0] == 0 and h["mask"][5] == 0
    # invariants: per bin with >= 2 valid genes z has mean 0 and sd 1; single-gene bin z == 1
    for b in range(20):
        zb = h["disp_norm"][h["bin"] == b]
        zb = zb[~np.isnan(zb)]
        if zb.size >= 2:
            assert abs(zb.mean()) < 1e-9 and abs(zb.std(ddof=1) - 1) < 1e-9
        elif zb.size == 1:
            assert zb[0] == 1.0


def _read_golden(path):
    cases, cur = [], {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line == "---":
            cases.append(cur); cur = {}
            continue
        k, v = line.split(":", 1)
        cur[k.strip()] = v.split()
    cases.append(cur)
    return cases


def test_hvg_hand_worked_golden():
    for c in _read_golden(os.path.join(HERE, "golden", "hvg_tiny.txt")):
        mean = np.array(c["mean"], float); var = np.array(c["var"], float)
        h = O.hvg_select(mean, var, int(c["n_top"][0]), int(c["n_bins"][0]), seurat_log=False)
        np.testing.assert_allclose(h["disp"], np.array(c["disp"], float), rtol=1e-15)
        np.testing.assert_allclose(h["edges"], np.array(c["edges"], float), rtol=1e-14)
        assert list(h["bin"]) == [int(x) for x in c["bin"]]
        np.testing.assert_allclose(h["disp_norm"], np.array(c["z"], float), rtol=1e-14, atol=1e-15)
        assert list(h["indices"]) == [int(x) for x in c["selected"]]
        assert h["count"] == len(c["selected"])


def test_hvg_edge_cases():
    # n_top larger than the number of valid genes -> all valid genes (reading R12)
    mean = np.array([1.0, 2.0, 0.0, 4.0]); var = np.array([2.0, 3.0, 0.0, 2.0])
    h = O.hvg_select(mean, var, 10, 2)
    assert h["count"] == 3 and h["mask"][2] == 0
    # literal single-gene rule: z = (d - 0)/d, so ln d == 0 gives 0/0 = NaN (not selected)
    h = O.hvg_select(mean, np.array([1.0, 3.0, 0.0, 2.0]), 10, 2)
    assert np.isnan(h["disp_norm"][0]) and h["count"] == 2
    # gene relabelling permutes the outputs
    rng = np.random.default_rng(3)
    mean = np.exp(rng.normal(0, 1, 200)); var = mean * np.exp(rng.normal(0, 0.5, 200))
    h0 = O.hvg_select(mean, var, 20, 20)
    p = rng.permutation(200)
    h1 = O.hvg_select(mean[p], var[p], 20, 20)
    np.testing.assert_allclose(h1["disp_norm"], h0["disp_norm"][p], rtol=1e-10, equal_nan=True)
    assert np.array_equal(h1["mask"], h0["mask"][p])
    assert h0["count"] == 20


def test_hvg_cutoffs_loops_and_special_windows():
    """NEXT-4 (part): window selection against explicit loops; infinite window == all non-NaN z."""
    rng = np.random.default_rng(3)
    m = rng.uniform(0, 4, 500); z = rng.normal(0, 1.5, 500); z[::17] = np.nan
    o = O.hvg_cutoffs(m, z)
    want = [j for j in range(500) if 0.0125 < m[j] < 3.0 and z[j] > 0.5 and not np.isnan(z[j])]
    assert o["indices"].tolist() == want and o["count"] == len(want) and o["mask"].sum() == len(want)
    o = O.hvg_cutoffs(m, z, -np.inf, np.inf, -np.inf, np.inf)
    assert o["count"] == int((~np.isnan(z)).sum())
    assert O.hvg_cutoffs(m, z, 1.0, 1.0)["count"] == 0              # empty (strict) window
    m2 = np.array([0.0125, 3.0, 1.0]); z2 = np.array([1.0, 1.0, 0.5])
    assert O.hvg_cutoffs(m2, z2)["count"] == 0                      # every bound is strict
