"""Pins for the NEXT-4 oracle functions hvg_cell_ranger and hvg_merge_batches: numpy.percentile,
pandas.cut / groupby restatements, invariants of the median / MAD normalisation, a hand-worked
fixture, and the special cases of the batch merge."""
import os

import numpy as np
import pandas as pd
import pytest

from oracle import oracle_np as O

HERE = os.path.dirname(os.path.abspath(__file__))


def _moments(G, seed, zeros=0):
    rng = np.random.default_rng(seed)
    mean = np.exp(rng.normal(-1.0, 1.5, G))
    var = mean * np.exp(rng.normal(0.3, 0.6, G))
    if zeros:
        idx = rng.choice(G, zeros, replace=False)
        mean[idx] = 0.0
        var[idx] = 0.0
    return mean, var


@pytest.mark.parametrize("n", [1, 2, 5, 21, 100, 1001])
def test_percentile_linear_is_numpy_percentile(n):
    rng = np.random.default_rng(n)
    a = np.sort(rng.lognormal(0, 2, n))
    for q in range(0, 105, 5):
        assert O.percentile_linear(a, q) == float(np.percentile(a, q)), (n, q)


@pytest.mark.parametrize("G,seed,zeros", [(400, 0, 0), (3000, 1, 0), (2000, 2, 150)])
def test_cell_ranger_against_pandas(G, seed, zeros):
    mean, var = _moments(G, seed, zeros)
    n_top = G // 10
    r = O.hvg_cell_ranger(mean, var, n_top)
    # independent restatement: numpy.percentile edges (duplicates dropped), pandas.cut, groupby
    m0 = mean.copy(); m0[m0 == 0] = 1e-12
    d = var / m0
    edges = np.unique(np.r_[-np.inf, np.percentile(mean, np.arange(10, 105, 5)), np.inf])
    codes = pd.cut(pd.Series(mean), edges, labels=False).to_numpy()
    assert np.array_equal(r["edges"], edges)
    assert np.array_equal(r["bin"], codes.astype(np.int32))
    df = pd.DataFrame({"d": d, "b": codes})
    med = df.groupby("b")["d"].median()
    mad = df.groupby("b")["d"].apply(lambda s: np.median(np.abs(s.to_numpy() - np.median(s.to_numpy()))) / 0.6744897501960817)
    with np.errstate(divide="ignore", invalid="ignore"):
        z = (d - med[codes].to_numpy()) / mad[codes].to_numpy()
    np.testing.assert_allclose(r["disp_norm"], z, rtol=1e-13, atol=0, equal_nan=True)
    zs = np.sort(z[~np.isnan(z)])[::-1]
    want = ~np.isnan(z) & (z >= zs[min(n_top, len(zs)) - 1])
    assert np.array_equal(r["mask"], want) and r["count"] >= min(n_top, len(zs))
    # invariants of the robust normalisation: per bin (>= 3 distinct values) median z = 0, median |z| = 0.6745
    for b in np.unique(codes):
        zb = r["disp_norm"][codes == b]
        zb = zb[np.isfinite(zb)]
        if len(zb) >= 3:
            assert abs(np.median(zb)) < 1e-12
            assert abs(np.median(np.abs(zb)) - 0.6744897501960817) < 1e-9


def test_cell_ranger_hand_worked_fixture():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "hvg_cell_ranger_tiny.txt")) if l.strip() and l[0] != "#"]
    mean = np.array([float(r[1]) for r in rows]); var = np.array([float(r[2]) for r in rows])
    r = O.hvg_cell_ranger(mean, var, 2)
    assert np.array_equal(r["disp"], [float(x[3]) for x in rows])
    assert np.array_equal(r["bin"], [int(x[4]) for x in rows])
    want_z = np.array([float(x[5]) for x in rows])
    np.testing.assert_allclose(r["disp_norm"], want_z, rtol=1e-15, atol=0, equal_nan=True)
    assert np.array_equal(r["mask"].astype(int), [int(x[6]) for x in rows])
    assert r["cutoff"] == 0.0 and r["count"] == 2


def test_cell_ranger_many_equal_means_merges_edges():
    mean = np.r_[np.zeros(60), np.arange(1, 41, dtype=float)]       # 60 % zeros: P10 .. P55 all equal 0
    var = np.r_[np.zeros(60), np.arange(1, 41, dtype=float) * 1.5]
    r = O.hvg_cell_ranger(mean, var, 5)
    assert len(r["edges"]) < 21 and np.all(np.diff(r["edges"]) > 0)
    assert np.all(r["bin"][:60] == 0) and r["count"] >= 0


def _pandas_merge(masks, z, n_top):
    B, G = masks.shape
    df = pd.DataFrame({"nb": masks.sum(axis=0), "zbar": np.nanmean(np.where(np.isnan(z), np.nan, z), axis=0)
                       if True else None})
    order = df.sort_values(["nb", "zbar"], ascending=False, na_position="last", kind="stable").index.to_numpy()
    return df, order


@pytest.mark.parametrize("B,G,seed", [(1, 300, 0), (3, 500, 1), (6, 800, 2)])
def test_merge_batches_against_pandas(B, G, seed):
    rng = np.random.default_rng(seed)
    z = rng.normal(0, 1, (B, G))
    z[rng.random((B, G)) < 0.1] = np.nan
    n_top = G // 8
    masks = np.zeros((B, G), dtype=bool)
    for b in range(B):
        zb = np.where(np.isnan(z[b]), -np.inf, z[b])
        masks[b, np.argsort(-zb)[:n_top]] = True
    import warnings
    with warnings.catch_warnings():
        warnings.simplefilter("ignore")
        df, order = _pandas_merge(masks, z, n_top)
    r = O.hvg_merge_batches(masks, z, n_top)
    assert np.array_equal(r["nbatches"], df["nb"].to_numpy())
    np.testing.assert_allclose(r["disp_norm_mean"], df["zbar"].to_numpy(), rtol=1e-13, equal_nan=True)
    top = set(order[:n_top].tolist())
    sel = set(np.nonzero(r["mask"])[0].tolist())
    assert top <= sel                                        # ties at the cutoff may add genes
    extra = sel - top
    c = order[n_top - 1]
    for j in extra:                                          # ... and only genes tied with the cutoff gene
        assert df["nb"][j] == df["nb"][c] and (df["zbar"][j] == df["zbar"][c] or (np.isnan(df["zbar"][j]) and np.isnan(df["zbar"][c])))
    if B == 1:                                               # one batch: its own selection, NaN-free part
        assert np.array_equal(r["mask"], masks[0])


def test_merge_batches_special_cases():
    # a gene selected in every batch outranks any gene selected in fewer, whatever its z
    masks = np.array([[1, 0, 1], [1, 1, 0]], dtype=bool)
    z = np.array([[-5.0, 9.0, 3.0], [-5.0, 9.0, np.nan]])
    r = O.hvg_merge_batches(masks, z, 1)
    assert r["mask"].tolist() == [True, False, False] and r["nbatches"].tolist() == [2, 1, 1]
    np.testing.assert_allclose(r["disp_norm_mean"], [-5.0, 9.0, 3.0])
    r2 = O.hvg_merge_batches(masks, z, 2)                    # genes 1 and 2 share nbatches = 1: higher zbar wins
    assert r2["mask"].tolist() == [True, True, False]
    zn = np.array([[np.nan, 1.0], [np.nan, 1.0]])
    r3 = O.hvg_merge_batches(np.zeros((2, 2), dtype=bool), zn, 2)    # cutoff in the NaN tail: the whole level
    assert r3["mask"].tolist() == [True, True] and np.isnan(r3["disp_norm_mean"][0])
