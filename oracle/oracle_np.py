"""CPU ORACLE — test infrastructure, NOT a product path.

Plain float64 / int64 NumPy restatement of the sparse-CSR preprocessing chain
of arxiv/paper_2603_02402 (rapids-singlecell): per-cell / per-gene QC,
normalize_total, log1p, per-gene moments and Seurat-flavour highly-variable-gene
selection.  Every function is the plain definition of what the step computes,
one pass per quantity, no blocking / fusion / reordering, so that it can be
checked against the paper by eye.  It shares no code with the CUDA path
(`paper_2603_02402_b200/csrc`) and imports nothing from the package.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this module.

Citations are `PAPER.md:L<line>` (the only reference file) plus the section.
Where the paper is silent the reading of DESIGN.md §3 (R1..R15) is followed
and named.

Pins (tests/test_oracle_*.py, `-m "not gpu"`):
  qc_metrics       dense brute force, scipy.sparse reductions, sum invariants
  normalize_total  row sums == target_sum, dense brute force, s == T identity
  log1p            numpy.log1p on the dense matrix, expm1 round trip, pattern kept
  gene_moments     np.mean / np.var(ddof) on the dense matrix, closed forms
  hvg_select       H3/H4 against pandas.cut; per-bin z mean 0 / sd 1; single-gene
                   bin => z == 1; brute-force loops on tiny inputs; hand-worked
                   fixture tests/golden/hvg_tiny.txt.
  filter_masks     thresholds written out; special cases (no threshold => keep all)
  subset_csr       dense brute force X[rows][:, cols], scipy.sparse fancy indexing,
                   identity / drop-all cases, nnz bookkeeping
  scale_dense      dense (X - mean) / sd with numpy; column mean 0 / sd 1 when unclipped;
                   zero-variance gene => sd 1; clip bounds; zero_center = False keeps zeros
  hvg_cutoffs      window tests written out with loops; infinite window == all non-NaN z
  gram_cov         numpy.cov of the dense matrix; explicit triple loop on tiny inputs; symmetry,
                   positive semi-definiteness; diag(C) == gene_moments' variance (ddof 1);
                   constant column => zero row / column of C; a gene permutation permutes C
  hvg_cell_ranger  percentile_linear == numpy.percentile; pandas.cut codes on the same edges;
                   pandas groupby median / MAD restatement; per-bin median of z == 0 and
                   median |z| == 0.6745; hand-worked fixture tests/golden/hvg_cell_ranger_tiny.txt
  hvg_merge_batches pandas sort_values([nbatches, zbar], ascending False, NaN last) restatement; one
                   batch == that batch's own selection; a gene selected everywhere outranks all
  pca_transform    (X - 1 mu^T) V on the dense centred matrix; columns of Z sum to 0 when mu is
                   the true mean; V = identity returns the centred matrix
  The CONSTANTS of H1/H5 (1e-12 floor, 0.1 % edge extension, ddof = 1 inside
  bins, z = 1 rule) are not in PAPER.md ("follows scanpy", L87) and scanpy is
  not installed: those constants are **parity unpinned** against the paper.
"""
from __future__ import annotations

import numpy as np

F32 = np.float32
F64 = np.float64
I64 = np.int64
I32 = np.int32


def _row_ids(indptr: np.ndarray) -> np.ndarray:
    """i(p): the row of every stored entry."""
    indptr = np.asarray(indptr, dtype=I64)
    n = indptr.shape[0] - 1
    return np.repeat(np.arange(n, dtype=I64), np.diff(indptr))


def _int_sum(groups: np.ndarray, values_i64: np.ndarray, size: int) -> np.ndarray:
    """Exact int64 group sums (float64 bincount is exact below 2**53)."""
    w = values_i64.astype(F64)
    out = np.bincount(groups, weights=w, minlength=size)
    assert np.all(np.abs(out) < 2.0 ** 53), "integer sum not exactly representable"
    return out.astype(I64)


# --------------------------------------------------------------------------
# Q1..Q4  QC metrics  ("QC metrics" cell-wise on CSR; L17/L21
# "filtering"; the list of metrics is reading R1)
# --------------------------------------------------------------------------
def qc_metrics(indptr, indices, data, n_genes: int, gene_flags=None) -> dict:
    """Per-cell and per-gene QC reductions.

    Q1  T_i  = sum_{p in row i} (int64) x_p                 total_counts
    Q2  N_i  = #{p in row i : x_p != 0}                      n_genes_by_counts
    Q3  M_i  = sum_{p in row i, flag[j(p)] != 0} (int64) x_p ; pct_i = 100 M_i / T_i
    Q4  C_j  = #{p : j(p) = j, x_p != 0} ;  T_j = sum_{p: j(p)=j} (int64) x_p
    "detected" means value != 0, not "stored" (R2).  T_i == 0 -> pct NaN (R3).
    Totals are int64 sums of the truncated values (R4).
    """
    indptr = np.asarray(indptr, dtype=I64)
    indices = np.asarray(indices, dtype=I64)
    data = np.asarray(data, dtype=F32)
    n = indptr.shape[0] - 1
    rows = _row_ids(indptr)
    xi = data.astype(F64).astype(I64)            # (int64) x_p, truncation
    nzmask = data != 0

    cell_total = _int_sum(rows, xi, n)
    cell_n_genes = np.bincount(rows[nzmask], minlength=n).astype(I32)
    if gene_flags is None:
        cell_flag_total = np.zeros(n, dtype=I64)
    else:
        fl = np.asarray(gene_flags) != 0
        sel = fl[indices]
        cell_flag_total = _int_sum(rows[sel], xi[sel], n)
    with np.errstate(divide="ignore", invalid="ignore"):
        pct = (100.0 * cell_flag_total.astype(F64) / cell_total.astype(F64)).astype(F32)

    gene_n_cells = np.bincount(indices[nzmask], minlength=n_genes).astype(I32)
    gene_total = _int_sum(indices, xi, n_genes)
    return dict(
        cell_total_i64=cell_total,
        cell_total_f32=cell_total.astype(F32),
        cell_n_genes=cell_n_genes,
        cell_flag_total_i64=cell_flag_total,
        cell_flag_pct=pct,
        gene_n_cells=gene_n_cells,
        gene_total_i64=gene_total,
    )


# --------------------------------------------------------------------------
# N1  normalize_total   PAPER.md:L91  x'_ij = (x_ij / sum_j x_ij) * s
# --------------------------------------------------------------------------
def normalize_total(indptr, data, target_sum: float, cell_total_i64=None):
    """Returns (x' as float32, scale float64[n]).

    scale_i = s / T_i in float64; x'_p = (float32)((double)x_p * scale_i): one
    rounding (R5).  A cell with T_i == 0 is left untouched, scale 1 (R3).
    When totals are not supplied they are the float64 row sums of the data.
    """
    indptr = np.asarray(indptr, dtype=I64)
    data = np.asarray(data, dtype=F32)
    n = indptr.shape[0] - 1
    rows = _row_ids(indptr)
    if cell_total_i64 is None:
        tot = np.bincount(rows, weights=data.astype(F64), minlength=n)
    else:
        tot = np.asarray(cell_total_i64).astype(F64)
    scale = np.ones(n, dtype=F64)
    ok = tot != 0
    scale[ok] = F64(target_sum) / tot[ok]
    out = (data.astype(F64) * scale[rows]).astype(F32)
    return out, scale


# --------------------------------------------------------------------------
# L1  log1p   PAPER.md:L91  x''_ij = log(1 + x'_ij), natural log (R7)
# --------------------------------------------------------------------------
def log1p(data):
    return np.log1p(np.asarray(data, dtype=F32).astype(F64)).astype(F32)


# --------------------------------------------------------------------------
# M1  per-gene moments   PAPER.md:L91 "per-gene mean and variance ... custom GPU
# reduction kernel that operates directly on sparse matrices"; L137.
# --------------------------------------------------------------------------
def gene_moments(indptr, indices, data, n_genes: int, transform: int = 0, ddof: int = 1):
    """mean_j, var_j over ALL n cells (zeros included), float64.

    v_p = x_p (transform 0) or expm1(x_p) (transform 1, reading R8).
    mean_j = (1/n) sum_p v_p ;
    var_j  = ( sum_{stored} (v_p - mean_j)^2 + (n - nnz_j) mean_j^2 ) / (n - ddof)
    i.e. the textbook two-pass variance of the dense column; ddof = 1 is the
    (n-1) convention the paper uses for its covariance (L95, reading R11).
    Returns (mean, var, S1, S2) with S1 = sum v, S2 = sum v^2.
    """
    indptr = np.asarray(indptr, dtype=I64)
    indices = np.asarray(indices, dtype=I64)
    n = indptr.shape[0] - 1
    v = np.asarray(data, dtype=F32).astype(F64)
    if transform == 1:
        v = np.expm1(v)
    elif transform != 0:
        raise ValueError("transform must be 0 or 1")
    s1 = np.bincount(indices, weights=v, minlength=n_genes)
    s2 = np.bincount(indices, weights=v * v, minlength=n_genes)
    stored = np.bincount(indices, minlength=n_genes).astype(F64)
    mean = s1 / F64(n) if n > 0 else np.zeros(n_genes)
    dev = v - mean[indices]
    ss = np.bincount(indices, weights=dev * dev, minlength=n_genes)
    ss = ss + (F64(n) - stored) * mean * mean
    with np.errstate(divide="ignore", invalid="ignore"):
        var = ss / F64(n - ddof)
    return mean, var, s1, s2


# --------------------------------------------------------------------------
# H1..H7  Seurat-flavour HVG selection.  PAPER.md:L91 "Highly variable gene
# selection is based on per-gene mean and variance"; L39 "gene selection"
# kernel; L87 "follow the algorithmic implementations of scanpy".  The steps
# are reading R8/R9/R10/R12; their constants are parity
# unpinned against PAPER.md (see module header).
# --------------------------------------------------------------------------
def bin_edges(m: np.ndarray, n_bins: int) -> np.ndarray:
    """H3: n_bins equal-width, right-closed bins over [min m, max m].

    step = (hi - lo)/n_bins ; edge_k = fl(fl(k*step) + lo) for k < n_bins ;
    edge_{n_bins} = hi ; then edge_0 -= 0.001*(hi - lo).
    Degenerate hi == lo (R10): lo -= 0.001*|lo| (or 0.001 when lo == 0),
    hi += 0.001*|hi| (or 0.001), no further extension.
    """
    m = np.asarray(m, dtype=F64)
    lo = F64(np.min(m))
    hi = F64(np.max(m))
    degenerate = lo == hi
    if degenerate:
        lo = lo - (F64(0.001) * abs(lo) if lo != 0 else F64(0.001))
        hi = hi + (F64(0.001) * abs(hi) if hi != 0 else F64(0.001))
    step = (hi - lo) / F64(n_bins)
    edges = np.empty(n_bins + 1, dtype=F64)
    for k in range(n_bins):
        edges[k] = F64(k) * step + lo       # two roundings, no fused multiply-add
    edges[n_bins] = hi
    if not degenerate:
        edges[0] = edges[0] - (hi - lo) * F64(0.001)
    return edges


def assign_bins(m: np.ndarray, edges: np.ndarray) -> np.ndarray:
    """H4: bin(m) = smallest k with m <= edge_{k+1}  (intervals (edge_k, edge_{k+1}])."""
    m = np.asarray(m, dtype=F64)
    nb = edges.shape[0] - 1
    out = np.empty(m.shape[0], dtype=I32)
    for g in range(m.shape[0]):
        k = 0
        while k < nb - 1 and not (m[g] <= edges[k + 1]):
            k += 1
        out[g] = k
    return out


def hvg_select(gene_mean, gene_var, n_top: int, n_bins: int = 20, seurat_log: bool = True) -> dict:
    """H1..H7.  Inputs: per-gene mean and variance (float64).

    H1  mean == 0 -> 1e-12 ;  d = var / mean
    H2  (seurat_log) d == 0 -> NaN ; d = ln d ; m = log1p(mean)
    H3/H4  20 equal-width bins over m, right-closed
    H5  per bin: mu_b = mean of the non-NaN d, sigma_b = their sample sd (ddof 1);
        exactly one non-NaN gene in the bin -> sigma_b = mu_b, mu_b = 0 (z = 1)
    H6  z = (d - mu_b) / sigma_b
    H7  cutoff = n_top-th largest non-NaN z (all of them if fewer, R12);
        mask = z >= cutoff (ties at the cutoff are all selected)
    """
    mean = np.array(gene_mean, dtype=F64, copy=True)
    var = np.asarray(gene_var, dtype=F64)
    G = mean.shape[0]
    mean[mean == 0] = F64(1e-12)
    with np.errstate(divide="ignore", invalid="ignore"):
        d = var / mean
        if seurat_log:
            d = np.where(d == 0, np.nan, d)
            d = np.log(d)
            m = np.log1p(mean)
        else:
            m = mean.copy()
    edges = bin_edges(m, n_bins)
    b = assign_bins(m, edges)

    mu_b = np.full(n_bins, np.nan)
    sd_b = np.full(n_bins, np.nan)
    for k in range(n_bins):
        dk = d[b == k]
        dk = dk[~np.isnan(dk)]
        if dk.shape[0] == 0:
            continue
        mk = np.sum(dk) / F64(dk.shape[0])
        if dk.shape[0] == 1:
            mu_b[k] = 0.0
            sd_b[k] = mk
        else:
            mu_b[k] = mk
            sd_b[k] = np.sqrt(np.sum((dk - mk) ** 2) / F64(dk.shape[0] - 1))
    with np.errstate(divide="ignore", invalid="ignore"):
        z = (d - mu_b[b]) / sd_b[b]

    valid = ~np.isnan(z)
    n_valid = int(valid.sum())
    k = min(int(n_top), n_valid)
    if k > 0:
        zs = np.sort(z[valid])[::-1]
        cutoff = zs[k - 1]
        mask = valid & (z >= cutoff)
    else:
        cutoff = np.nan
        mask = np.zeros(G, dtype=bool)
    idx = np.nonzero(mask)[0].astype(I32)
    return dict(mean_t=m, disp=d, disp_norm=z, bin=b, edges=edges,
                mask=mask.astype(np.uint8), indices=idx, count=int(idx.shape[0]),
                cutoff=cutoff)


# --------------------------------------------------------------------------
# The chain as the paper orders it (QC -> normalize ->
# log1p -> HVG).  Composition only; no arithmetic of its own.
# --------------------------------------------------------------------------
def preprocess_chain(indptr, indices, data, n_genes, gene_flags, target_sum, n_top,
                     n_bins=20, ddof=1, hvg_on="linear") -> dict:
    qc = qc_metrics(indptr, indices, data, n_genes, gene_flags)
    xn, scale = normalize_total(indptr, data, target_sum, qc["cell_total_i64"])
    xl = log1p(xn)
    mean_log, var_log, _, _ = gene_moments(indptr, indices, xl, n_genes, 0, ddof)
    mean_lin, var_lin, _, _ = gene_moments(indptr, indices, xn, n_genes, 0, ddof)
    if hvg_on == "linear":
        hv = hvg_select(mean_lin, var_lin, n_top, n_bins)
    else:
        hv = hvg_select(mean_log, var_log, n_top, n_bins)
    return dict(qc=qc, x_norm=xn, x_log=xl, mean_log=mean_log, var_log=var_log,
                mean_lin=mean_lin, var_lin=var_lin, hvg=hv)


# --------------------------------------------------------------------------- NEXT-1: filtering
def filter_masks(qc: dict, min_genes: int = 0, min_counts: int = 0, max_pct_flag: float = np.inf,
                 min_cells: int = 0, min_gene_counts: int = 0):
    """Cell and gene keep-masks from the QC outputs ("filtering"; the
    thresholds are scanpy's filter_cells / filter_genes arguments, named in SURVEY.md §8(f)
    NEXT-1; the paper states none).  A cell is kept when it has >= min_genes detected genes,
    >= min_counts total counts and <= max_pct_flag percent of its counts in the flagged set
    (a NaN percentage -- an empty cell -- fails any finite max_pct_flag); a gene is kept when
    it is detected in >= min_cells cells and has >= min_gene_counts total counts."""
    pct = np.asarray(qc["cell_flag_pct"], F64)
    cell = (np.asarray(qc["cell_n_genes"], I64) >= min_genes) & \
           (np.asarray(qc["cell_total_i64"], I64) >= min_counts)
    if np.isfinite(max_pct_flag):
        cell &= pct <= max_pct_flag                     # NaN <= x is False
    gene = (np.asarray(qc["gene_n_cells"], I64) >= min_cells) & \
           (np.asarray(qc["gene_total_i64"], I64) >= min_gene_counts)
    return cell.astype(np.uint8), gene.astype(np.uint8)


def subset_csr(indptr, indices, data, n_genes: int, keep_rows, keep_cols):
    """X[keep_rows][:, keep_cols] as a new CSR (filter_cells /
    filter_genes / HVG column subsetting = row and column removal with a rebuilt int64
    indptr).  Kept columns are renumbered in ascending order (new index = number of kept
    columns before it); the stored entries of a kept row keep their order and values; explicit
    zeros stay stored.  Plain loop over the rows."""
    indptr = np.asarray(indptr, I64)
    indices = np.asarray(indices, I32)
    data = np.asarray(data, F32)
    keep_rows = np.asarray(keep_rows).astype(bool)
    keep_cols = np.asarray(keep_cols).astype(bool)
    assert keep_rows.shape == (len(indptr) - 1,) and keep_cols.shape == (n_genes,)
    col_map = np.full(n_genes, -1, dtype=I64)
    col_map[keep_cols] = np.arange(int(keep_cols.sum()), dtype=I64)
    out_ptr = [0]
    out_idx, out_val = [], []
    for i in np.nonzero(keep_rows)[0]:
        lo, hi = int(indptr[i]), int(indptr[i + 1])
        j = col_map[indices[lo:hi]]
        sel = j >= 0
        out_idx.append(j[sel].astype(I32))
        out_val.append(data[lo:hi][sel])
        out_ptr.append(out_ptr[-1] + int(sel.sum()))
    idx = np.concatenate(out_idx) if out_idx else np.zeros(0, I32)
    val = np.concatenate(out_val) if out_val else np.zeros(0, F32)
    return np.asarray(out_ptr, I64), idx.astype(I32), val.astype(F32), int(keep_cols.sum())


# --------------------------------------------------------------------------- NEXT-3 (first half): scale
def scale_dense(indptr, indices, data, n_genes: int, gene_mean, gene_var, max_value=None,
                zero_center: bool = True):
    """z-score per gene, optionally clipped ("scaling"; SURVEY.md §8(f)
    NEXT-3 "scale: z-score using the log-scale moments already produced").  Dense float32
    [n_rows, n_genes] output:  y_ij = (x_ij - mean_j) / sd_j  with sd_j = sqrt(var_j) and
    sd_j = 1 where var_j == 0 (reading R16: scanpy's convention; the paper gives
    none); zero_center = False divides only (zeros stay zero).  max_value: clip to
    [-max_value, max_value] when centred, to (-inf, max_value] otherwise (R16)."""
    indptr = np.asarray(indptr, I64)
    n = len(indptr) - 1
    mean = np.asarray(gene_mean, F64)
    sd = np.sqrt(np.asarray(gene_var, F64))
    sd = np.where(sd == 0.0, 1.0, sd)
    dense = np.zeros((n, n_genes), dtype=F64)
    rows = _row_ids(indptr)
    dense[rows, np.asarray(indices, I64)] = np.asarray(data, F64)
    y = (dense - mean[None, :]) / sd[None, :] if zero_center else dense / sd[None, :]
    if max_value is not None:
        y = np.clip(y, -max_value if zero_center else -np.inf, max_value)
    return y.astype(F32)


# --------------------------------------------------------------------------- NEXT-4 (part): cutoffs
def hvg_cutoffs(mean_t, disp_norm, min_mean=0.0125, max_mean=3.0, min_disp=0.5, max_disp=np.inf):
    """Threshold-based HVG selection (SURVEY.md §8(f) NEXT-4 "threshold-based selection
    (mean/dispersion windows)"): from the transformed mean m and the normalised dispersion z of
    hvg_select, gene j is selected when  min_mean < m_j < max_mean  and  min_disp < z_j <
    max_disp  (strict; a NaN z fails).  The defaults and the strictness are scanpy's (the paper
    gives none: parity unpinned against PAPER.md, reading R17)."""
    m = np.asarray(mean_t, F64)
    z = np.asarray(disp_norm, F64)
    with np.errstate(invalid="ignore"):
        mask = (m > min_mean) & (m < max_mean) & (z > min_disp) & (z < max_disp)
    return dict(mask=mask.astype(np.uint8), indices=np.nonzero(mask)[0].astype(I32), count=int(mask.sum()))


# ---------------------------------------------------------------------------- NEXT-3, second half
def gram_cov(indptr, indices, data, n_genes: int) -> dict:
    """Sparse PCA front end, "Principal component analysis": for X in R^{n x p}
    (cells x genes, CSR)
        mu = (1/n) X^T 1                       per-feature means
        S  = X^T X                             Gram matrix (the paper accumulates the upper
                                               triangle and mirrors it; here all of it, plainly)
        C  = (1/(n-1)) (S - n mu mu^T)         mean-centred covariance, no explicit centring
    in float64 from the float32 values.  Returns {"mean": [p], "gram": [p, p], "cov": [p, p]}.
    n must be >= 2 (the 1/(n-1) of L95).  S is formed by definition, entry by entry of the sparse
    rows: S[a, b] = sum over cells i of x_ia x_ib (a dense matmul of the densified matrix is the
    library step that evaluates exactly this sum)."""
    indptr = np.asarray(indptr, dtype=I64)
    indices = np.asarray(indices, dtype=I64)
    n = indptr.shape[0] - 1
    assert n >= 2, "covariance needs at least two cells"
    X = np.zeros((n, n_genes), dtype=F64)
    X[_row_ids(indptr), indices] = np.asarray(data, dtype=F32).astype(F64)
    mu = X.sum(axis=0) / n
    S = X.T @ X
    C = (S - n * np.outer(mu, mu)) / (n - 1)
    return {"mean": mu, "gram": S, "cov": C}


def pca_transform(indptr, indices, data, n_genes: int, V, mean) -> np.ndarray:
    """PAPER.md:L95  Z = X V - 1 (mu^T V): the sparse-to-dense projection with implicit centring
    (V in R^{p x k} the loadings, mu the per-feature means).  float64; returns Z [n, k]."""
    indptr = np.asarray(indptr, dtype=I64)
    indices = np.asarray(indices, dtype=I64)
    V = np.asarray(V, dtype=F64)
    mean = np.asarray(mean, dtype=F64)
    n = indptr.shape[0] - 1
    X = np.zeros((n, n_genes), dtype=F64)
    X[_row_ids(indptr), indices] = np.asarray(data, dtype=F32).astype(F64)
    return X @ V - np.ones((n, 1)) * (mean @ V)[None, :]


# ---------------------------------------------------------------------------- NEXT-4: other HVG variants
MAD_SCALE = 0.6744897501960817          # Phi^-1(3/4): MAD / MAD_SCALE estimates sigma for normal data


def percentile_linear(sorted_vals: np.ndarray, q_percent: float) -> float:
    """Linear-interpolation percentile of an ascending array (the textbook definition numpy's
    default method evaluates): virtual index vi = (q / 100) (n - 1), lo = floor(vi), t = vi - lo,
    value = a[lo] + (a[hi] - a[lo]) t for t < 0.5, else a[hi] - (a[hi] - a[lo]) (1 - t)
    (the second form keeps the result exact at t -> 1), with separate multiply and add."""
    a = np.asarray(sorted_vals, dtype=F64)
    n = a.shape[0]
    vi = (F64(q_percent) / F64(100.0)) * F64(n - 1)
    lo = int(np.floor(vi))
    hi = min(lo + 1, n - 1)
    t = F64(vi - F64(lo))
    diff = F64(a[hi] - a[lo])
    if t < 0.5:
        return float(F64(a[lo] + F64(diff * t)))
    return float(F64(a[hi] - F64(diff * F64(F64(1.0) - t))))


def hvg_cell_ranger(gene_mean, gene_var, n_top: int) -> dict:
    """Cell-ranger-flavour HVG selection ("Highly variable gene
    selection is based on per-gene mean and variance", L87 "follow the algorithmic implementations
    of scanpy"; the paper gives no constants -- DESIGN.md reading R18, parity unpinned against
    PAPER.md).  Input: mean / variance of the NORMALISED, non-logged matrix x'.
      C1  mean == 0 -> 1e-12;  d = var / mean               (no log transforms)
      C2  edges = -inf, P10, P15, .., P100 of the means (linear interpolation), +inf;
          equal edges are merged (an empty interval holds no gene)
      C3  bin(m) = the interval (e_k, e_{k+1}] that holds m  (right-closed)
      C4  per bin: med_b = median of the d in the bin, mad_b = median |d - med_b| / 0.6745
      C5  z = (d - med_b) / mad_b                            (IEEE: mad_b = 0 gives +-inf or NaN)
      C6  cutoff = n_top-th largest non-NaN z; mask = z is not NaN and z >= cutoff (as H7)
    Returns disp, disp_norm, bin (index into the merged edges), edges, mask, cutoff, count."""
    mean = np.asarray(gene_mean, dtype=F64).copy()
    var = np.asarray(gene_var, dtype=F64)
    G = mean.shape[0]
    mean0 = mean.copy()
    mean0[mean0 == 0] = 1e-12
    d = var / mean0
    srt = np.sort(mean)
    edges = [-np.inf] + [percentile_linear(srt, q) for q in range(10, 105, 5)] + [np.inf]
    merged = [edges[0]]
    for e in edges[1:]:
        if e != merged[-1]:
            merged.append(e)
    edges = np.asarray(merged, dtype=F64)
    nb = edges.shape[0] - 1
    bins = np.empty(G, dtype=I32)
    for j in range(G):
        k = 0
        while not (mean[j] <= edges[k + 1]):              # smallest k with m <= e_{k+1}
            k += 1
        bins[j] = k
    med = np.full(nb, np.nan)
    mad = np.full(nb, np.nan)
    for b in range(nb):
        sel = (bins == b) & ~np.isnan(d)
        if sel.any():
            med[b] = np.median(d[sel])
            mad[b] = np.median(np.abs(d[sel] - med[b])) / MAD_SCALE
    with np.errstate(divide="ignore", invalid="ignore"):
        z = (d - med[bins]) / mad[bins]
    valid = ~np.isnan(z)
    k = min(int(n_top), int(valid.sum()))
    if k > 0:
        cutoff = np.sort(z[valid])[::-1][k - 1]
        mask = valid & (z >= cutoff)
    else:
        cutoff = np.nan
        mask = np.zeros(G, dtype=bool)
    return {"disp": d, "disp_norm": z, "bin": bins, "edges": edges, "median": med, "mad": mad,
            "mask": mask, "cutoff": cutoff, "count": int(mask.sum()),
            "indices": np.nonzero(mask)[0].astype(I32)}


def hvg_merge_batches(masks, disp_norm, n_top: int) -> dict:
    """Per-batch HVG (reading R19, scanpy's batch_key convention, parity
    unpinned against PAPER.md): the selection runs per batch; then per gene
      B1  nbatches_j = number of batches that selected gene j
      B2  zbar_j = mean over the batches of the gene's non-NaN normalised dispersions (NaN if none)
      B3  genes are ranked by (nbatches, zbar) descending, NaN zbar last within its nbatches level;
          the n_top-th gene of that order sets the cutoff pair and every gene at or above it is
          selected (ties at the cutoff select more than n_top, as H7).
    masks: bool [B, G]; disp_norm: float64 [B, G]."""
    masks = np.asarray(masks).astype(bool)
    z = np.asarray(disp_norm, dtype=F64)
    Bn, G = masks.shape
    nbat = masks.sum(axis=0).astype(I32)
    cnt = (~np.isnan(z)).sum(axis=0)
    zs = np.where(np.isnan(z), 0.0, z).sum(axis=0)        # batch order 0 .. B-1: a fixed summation order
    zbar = np.where(cnt > 0, zs / np.maximum(cnt, 1), np.nan)
    k = min(int(n_top), G)
    # rank: nbatches descending, NaN zbar last within a level, then zbar descending
    order = sorted(range(G), key=lambda j: (-int(nbat[j]), bool(np.isnan(zbar[j])),
                                            0.0 if np.isnan(zbar[j]) else -zbar[j]))
    if k > 0:
        c = order[k - 1]
        cn, cz, cnan = int(nbat[c]), zbar[c], bool(np.isnan(zbar[c]))
        mask = np.zeros(G, dtype=bool)
        for j in range(G):
            if nbat[j] > cn:
                mask[j] = True
            elif nbat[j] == cn:
                if cnan:
                    mask[j] = True                        # the cutoff sits in the NaN tail of its level
                else:
                    mask[j] = (not np.isnan(zbar[j])) and zbar[j] >= cz
    else:
        mask = np.zeros(G, dtype=bool)
    return {"nbatches": nbat, "disp_norm_mean": zbar, "mask": mask, "count": int(mask.sum()),
            "indices": np.nonzero(mask)[0].astype(I32)}
