/*
 * rsc.h — C ABI of librsc_b200: the sparse-CSR single-cell preprocessing chain of
 * arxiv/paper_2603_02402 (rapids-singlecell) as hand-written sm_100a CUDA kernels.
 *
 * The chain (PAPER.md:L47, L145 workflow order; L85 "CSR format is used for
 * cell-wise operations (e.g., normalization, QC metrics)"; L91 "Preprocessing and
 * normalization"):
 *     QC reductions -> normalize_total -> log1p -> per-gene moments -> HVG selection
 *
 * Conventions (all entry points)
 *   - Pointers are DEVICE pointers owned by the caller unless the name says `host`.
 *     The library never allocates or frees device memory and never synchronises
 *     the stream: every call only enqueues work on `stream` (a cudaStream_t passed
 *     as void*; NULL = the legacy default stream) and returns.
 *   - Scratch memory comes from the caller: `ws` must hold at least the number of
 *     bytes the matching `*_workspace_bytes` query returns and be 256-byte aligned.
 *     Its contents are undefined on entry and on exit.
 *   - Return value: RSC_OK or a negative rsc_status.  After a failure
 *     rsc_last_error() returns a thread-local, human-readable description.
 *     Arguments are validated on the host; the matrix CONTENT is not validated
 *     (canonical CSR is a precondition: indptr non-decreasing with indptr[0]=0 and
 *     indptr[n_rows]=nnz, 0 <= indices < n_cols, no duplicate column inside a row).
 *   - Optional outputs may be NULL and are then skipped.
 *   - Matrix layout: float32 `data`, int32 `indices`, int64 `indptr`
 *     (BASELINE.json north_star; int64 lifts the ~2^31 nnz ceiling of PAPER.md:L43,
 *     L141).
 */
#ifndef RSC_H_
#define RSC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  RSC_OK = 0,
  RSC_ERR_INVALID_ARG = -1, /* NULL required pointer, negative size, bad parameter   */
  RSC_ERR_WORKSPACE = -2,   /* workspace too small or misaligned                     */
  RSC_ERR_CUDA = -3,        /* CUDA runtime / launch error (text in rsc_last_error)  */
  RSC_ERR_UNSUPPORTED = -4  /* current device is not compute capability 10.x         */
} rsc_status;

/* rsc_csr.flags */
#define RSC_CSR_SORTED 1 /* column indices strictly ascending inside every row.  Enables the
                            conflict-free shared-memory accumulation path; without it the
                            kernels fall back to L2 atomics (same results, slower).          */

typedef struct {
  int64_t n_rows;        /* cells n                                                   */
  int32_t n_cols;        /* genes G                                                   */
  int32_t flags;         /* RSC_CSR_* bits                                            */
  int64_t nnz;           /* == indptr[n_rows]; passed by the caller to avoid a sync   */
  const int64_t* indptr; /* [n_rows + 1]                                              */
  const int32_t* indices;/* [nnz]                                                     */
  float* data;           /* [nnz]; rewritten in place by normalize / log1p / fused    */
} rsc_csr;

/* Row split table (used by the streaming kernels to cut the gene axis into groups whose
 * accumulators fit one SM's shared memory).  Columns are cut into K = ceil(n_cols /
 * RSC_SPLIT_WIDTH) blocks; the table holds, for every row, K + 1 uint32 values
 *     splits[row * (K + 1) + k] = #{stored entries of the row with column < k * RSC_SPLIT_WIDTH}
 * (so splits[row][0] = 0 and splits[row][K] = the row length).  It is only meaningful for
 * rows with ascending column indices (RSC_CSR_SORTED).  rsc_qc_metrics can emit it while it
 * streams the matrix (binary searches in the row it has just read; rsc_qc_metrics_splits emits
 * only chosen entries, which is cheaper); rsc_row_splits computes it on its own. */
#define RSC_SPLIT_SHIFT 10
#define RSC_SPLIT_WIDTH (1 << RSC_SPLIT_SHIFT)
/* number of uint32 elements of the table */
size_t rsc_row_splits_count(int64_t n_rows, int32_t n_cols);
int rsc_row_splits(const rsc_csr* X, uint32_t* row_splits, void* stream);

const char* rsc_last_error(void);
/* Library version, "major.minor.patch". */
const char* rsc_version(void);
/* Number of CUDA kernels this library has launched so far in the calling process (host-side
 * counter; memsets / memcpys are not counted).  Used by bench.py to report gpu_launches. */
uint64_t rsc_kernel_launch_count(void);
/* Process-wide tuning / testing knobs (not needed in normal use; defaults in brackets):
 *   "fused_row_budget" [256]   rows a CTA of the fused pass takes between two checks of its
 *                              integer accumulator tables (1..256, rounded down to a power of
 *                              two); a check moves the genes whose words are half full to the
 *                              global totals
 *   "flush_all"        [0]     1 = every check moves EVERY gene (testing the exchange path)
 *   "qc_row_budget"    [512]   the same for the QC pass's packed count | total words (1..512)
 *   "grid_ctas"        [0]     CTAs of the streaming kernels, 0 = one per SM
 *   "force_generic"    [0]     1 = always take the generic L2-atomic kernels
 *   "host_chunk_nnz"   [150e6] rsc_preprocess_host: stored entries per pipelined row chunk (at most 16
 *                              chunks; 0 = one chunk: copy in, compute, copy out one after the other)
 *   "single_pass"      [0]     1 = rsc_preprocess runs QC + normalise + log1p + log-scale moments as ONE pass
 *                              over the matrix (pairs of CTAs exchanging the rows' partial totals through
 *                              distributed shared memory: 12 B / nnz of DRAM traffic instead of 20) when it
 *                              can: sorted rows, 16-byte aligned arrays, 512 <= n_cols <= 32 768,
 *                              n_rows < 2^24, which_moments == RSC_MOMENTS_LOG.  Same results (integers and
 *                              x'' bit for bit); slower than the default two passes on B200
 *   "hvg_single_cta"   [0]     1 = rsc_hvg_select on its one-CTA kernel (default: a cluster of 8 CTAs
 *                              when n_bins <= 32 and n_genes <= 65 536)
 * Returns RSC_ERR_INVALID_ARG for an unknown key or a value out of range. */
int rsc_set_option(const char* key, long long value);

/* ---------------------------------------------------------------------------------
 * rsc_qc_metrics — per-cell and per-gene QC reductions.
 * PAPER.md:L85 ("QC metrics", cell-wise on CSR), L17/L21 ("filtering"); the list of
 * metrics is BASELINE.json north_star's (reading R1).
 *   cell_total_i64[i]      T_i = sum over row i of (int64) x          (exact integer)
 *   cell_total_f32[i]      (float) T_i
 *   cell_n_genes[i]        #{stored entries of row i with x != 0}
 *   cell_flag_total_i64[i] M_i = sum over row i, gene_flags[col] != 0, of (int64) x
 *   cell_flag_pct[i]       (float)(100.0 * M_i / T_i) evaluated in double; NaN when T_i = 0
 *   gene_n_cells[j]        #{stored entries of column j with x != 0}
 *   gene_total_i64[j]      sum over column j of (int64) x
 * Values are truncated to integers before summation; counts must be < 2^24.
 * gene_flags: uint8[n_cols] or NULL (then M_i = 0, pct = 0 or NaN).
 * row_splits: optional uint32[rsc_row_splits_count(n_rows, n_cols)] receiving the row split
 *   table (see above); written only when X->flags has RSC_CSR_SORTED, else left untouched.
 * Outputs are fully overwritten (no accumulation into previous contents).
 * ------------------------------------------------------------------------------- */
size_t rsc_qc_metrics_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);
int rsc_qc_metrics(const rsc_csr* X, const uint8_t* gene_flags,
                   int64_t* cell_total_i64, float* cell_total_f32, int32_t* cell_n_genes,
                   int64_t* cell_flag_total_i64, float* cell_flag_pct,
                   int32_t* gene_n_cells, int64_t* gene_total_i64, uint32_t* row_splits,
                   void* ws, size_t ws_bytes, void* stream);
/* The same call, but only the row_splits entries whose block index k is listed in
 * split_blocks (a HOST array of n_split_blocks <= 32 indices in [0, K]) are written; the other
 * entries of the table are left untouched.  The fused pass reads just a few entries per row
 * (rsc_moments_split_blocks tells which), and emitting only those spares the QC pass most of
 * the table's cost.  n_split_blocks = 0 -> the full table, as rsc_qc_metrics. */
int rsc_qc_metrics_splits(const rsc_csr* X, const uint8_t* gene_flags,
                          int64_t* cell_total_i64, float* cell_total_f32, int32_t* cell_n_genes,
                          int64_t* cell_flag_total_i64, float* cell_flag_pct,
                          int32_t* gene_n_cells, int64_t* gene_total_i64, uint32_t* row_splits,
                          const int32_t* split_blocks, int32_t n_split_blocks,
                          void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_normalize_total — PAPER.md:L91  x'_ij = (x_ij / sum_j x_ij) * s, in place.
 *   scale_i = target_sum / (float) T_i  (float32 division), data[p] *= scale_i.
 *   cell_total_i64: T_i from rsc_qc_metrics, or NULL -> the kernel sums each row
 *   itself (double accumulation of the float values).
 *   A row with T_i == 0 is left untouched (scale 1).
 *   cell_scale_out: optional float[n_rows] receiving scale_i.
 *   target_sum must be finite and > 0.
 * ------------------------------------------------------------------------------- */
int rsc_normalize_total(rsc_csr* X, float target_sum, const int64_t* cell_total_i64,
                        float* cell_scale_out, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_log1p — PAPER.md:L91  x''_ij = log(1 + x'_ij) (natural log), in place on
 * X->data; indptr / indices are not touched, log1p(0) = 0 keeps the pattern.
 * ------------------------------------------------------------------------------- */
int rsc_log1p(rsc_csr* X, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_gene_moments — PAPER.md:L91 / L137 "per-gene reduction kernels for mean and
 * variance" operating directly on the sparse matrix (no CSC copy, cf. L85).
 *   v = data[p] (transform 0) or expm1((double)data[p]) (transform 1)
 *   S1_j = sum v, S2_j = sum v^2 in double precision over the stored entries,
 *   mean_j = S1_j / n,  var_j = max(0, (S2_j - n mean_j^2) / (n - ddof)); zeros are
 *   included through n.  ddof in {0, 1}; n - ddof must be > 0.
 *   gene_sum / gene_sumsq: optional double[n_cols] receiving S1 / S2.
 * ------------------------------------------------------------------------------- */
size_t rsc_gene_moments_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);
int rsc_gene_moments(const rsc_csr* X, int transform, int ddof,
                     double* gene_mean, double* gene_var,
                     double* gene_sum, double* gene_sumsq,
                     void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_normalize_log1p_moments — the fused pass (BASELINE.json north_star; not in the
 * paper, which runs L91's three steps as separate kernels): every stored entry is
 * read once, x' = x * scale_i, x'' = log1p(x') is written back, and the per-gene
 * sums of the ROUNDED float32 x'' (log scale) and/or x' (linear scale) are
 * accumulated in double precision.
 *   which_moments: bit0 RSC_MOMENTS_LOG -> mean_log/var_log, bit1 RSC_MOMENTS_LIN ->
 *   mean_lin/var_lin (the matching pointers are then required).  By default the sums are
 *   accumulated on chip as EXACT integers (every value v is scaled by a power of two chosen on
 *   the device from the largest cell total, so that v * 2^k is an integer; S1 in 64 bits, S2
 *   in 96 bits, order-independent); values more than 2^19 times smaller
 *   than target_sum's binade, negative values and NaNs are added to the global double sums
 *   directly (same result, slower).  bit2 RSC_MOMENTS_FP64_ACC selects double-precision
 *   shared-memory accumulators instead (any value range, slower).
 *   X->indices and X->data must be 16-byte aligned for the streaming kernel (else the generic
 *   kernel serves the call: same results).
 *   row_splits: optional row split table of X (from rsc_qc_metrics / rsc_row_splits; a partial
 *   table from rsc_qc_metrics_splits must hold the entries rsc_moments_split_blocks lists for
 *   THIS n_cols and which_moments -- other entries are not read);
 *   NULL -> computed into the workspace when needed.
 *   cell_total_i64 is required (from rsc_qc_metrics).
 *   gene_n_cells: optional hint (from rsc_qc_metrics) used to balance the gene
 *   ranges of the shared-memory accumulators; results do not depend on it.
 *   gene_sums_out: optional double[4 * n_cols] receiving the raw sums
 *   S1log | S2log | S1lin | S2lin (n_cols each; only the requested sets are written).
 *   Row-sharded multi-GPU runs all-reduce these and call rsc_moments_finalize.
 * ------------------------------------------------------------------------------- */
#define RSC_MOMENTS_LOG 1
#define RSC_MOMENTS_LIN 2
#define RSC_MOMENTS_FP64_ACC 4
size_t rsc_normalize_log1p_moments_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);
/* Block indices k of the row split table that rsc_normalize_log1p_moments reads for this
 * n_cols / which_moments (the edges of its gene-range groups), written to blocks_out[0..cap);
 * returns their number (0 when the call would not use a table; > cap -> nothing written). */
int32_t rsc_moments_split_blocks(int32_t n_cols, int which_moments, int32_t* blocks_out, int32_t cap);
int rsc_normalize_log1p_moments(rsc_csr* X, float target_sum, const int64_t* cell_total_i64,
                                const int32_t* gene_n_cells, const uint32_t* row_splits,
                                int which_moments, int ddof,
                                double* mean_log, double* var_log,
                                double* mean_lin, double* var_lin, double* gene_sums_out,
                                void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_moments_finalize — mean_j = S1_j / n, var_j = max(0, (S2_j - n mean_j^2)/(n - ddof))
 * from raw per-gene sums (the last step of PAPER.md:L91's mean / variance kernel, split
 * out so that sums from several row shards (L141: chunks along the cell axis) can be
 * added first).  n_rows_total is the number of cells over ALL shards.
 * ------------------------------------------------------------------------------- */
int rsc_moments_finalize(int32_t n_genes, int64_t n_rows_total, int ddof, const double* S1,
                         const double* S2, double* gene_mean, double* gene_var, void* stream);

/* ---------------------------------------------------------------------------------
 * filtering and subsetting ("filtering"; the
 * workflow's filter_cells / filter_genes / HVG column subsetting steps, L47).
 *
 * rsc_filter_masks: uint8 keep-masks from the QC outputs.  A cell is kept when
 *   cell_n_genes >= min_genes, cell_total_i64 >= min_counts and cell_flag_pct <= max_pct_flag
 *   (a NaN percentage fails; max_pct_flag = +inf switches the test off); a gene is kept when
 *   gene_n_cells >= min_cells and gene_total_i64 >= min_gene_counts.  A NULL input array
 *   switches its test off; a NULL output mask is not computed.
 *
 * rsc_subset_csr_plan / rsc_subset_csr_fill: X[keep_rows][:, keep_cols] as a new CSR.  Kept
 *   columns are renumbered in ascending order; kept entries keep their order and values
 *   (explicit zeros stay stored); NULL mask = keep all.  plan writes out_indptr (capacity
 *   n_rows + 1, the first out_counts[0] + 1 entries are valid) and out_counts = {kept rows,
 *   kept columns, kept entries} (device int64[3]); the caller reads out_counts (its one
 *   synchronisation), allocates out_indices / out_data of out_counts[2] elements and calls
 *   fill with the SAME workspace (it holds the column map and the row offsets).
 * ------------------------------------------------------------------------------- */
typedef struct {
  int32_t min_genes;        /* cells: detected genes              */
  int32_t min_cells;        /* genes: cells detected in           */
  int64_t min_counts;       /* cells: total counts                */
  int64_t min_gene_counts;  /* genes: total counts                */
  float max_pct_flag;       /* cells: percent in the flagged set; +inf = off */
  int32_t pad;
} rsc_filter_params;
int rsc_filter_masks(int64_t n_rows, int32_t n_cols, const int32_t* cell_n_genes,
                     const int64_t* cell_total_i64, const float* cell_flag_pct,
                     const int32_t* gene_n_cells, const int64_t* gene_total_i64,
                     const rsc_filter_params* prm, uint8_t* cell_keep, uint8_t* gene_keep,
                     void* stream);
size_t rsc_subset_csr_workspace_bytes(int64_t n_rows, int32_t n_cols);
int rsc_subset_csr_plan(const rsc_csr* X, const uint8_t* keep_rows, const uint8_t* keep_cols,
                        int64_t* out_indptr, int64_t* out_counts, void* ws, size_t ws_bytes,
                        void* stream);
int rsc_subset_csr_fill(const rsc_csr* X, const uint8_t* keep_rows, int32_t* out_indices,
                        float* out_data, void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_hvg_cutoffs: threshold-based HVG selection from the
 * outputs of rsc_hvg_select (out_mean_t = m, out_disp_norm = z): gene j is selected when
 * min_mean < m_j < max_mean and min_disp < z_j < max_disp (strict; a NaN z fails; use
 * -inf / +inf to switch a bound off).  out_mask uint8[n_genes] and out_count int32[1] are
 * required; out_indices int32[n_genes] (selected genes, ascending) is optional.
 * ------------------------------------------------------------------------------- */
int rsc_hvg_cutoffs(int32_t n_genes, const double* mean_t, const double* disp_norm,
                    double min_mean, double max_mean, double min_disp, double max_disp,
                    uint8_t* out_mask, int32_t* out_indices, int32_t* out_count, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_pca_transform -- PAPER.md:L95 "The sparse-to-dense transform applies implicit centering in
 * chunks: Z = XV - 1 (mu^T V)": the projection of the cells on k loadings (the eigenvectors of C,
 * computed by the caller's eigensolver -- a library call, out of scope here).
 *   V: double[n_cols][n_comps] row-major; gene_mean: double[n_cols] (out_mean of rsc_gram_cov) or
 *   NULL (no centring: the uncentred truncated-SVD projection the paper also provides);
 *   out: float[n_rows][n_comps].  Products are accumulated in double from a float32 copy of V
 *   (|Z - Z_exact| <= 1e-7 * sum_j |x_ij V_jc| + float32 rounding of the result).
 *   1 <= n_comps <= 128.  ws: rsc_pca_transform_workspace_bytes(n_cols, n_comps).
 * ------------------------------------------------------------------------------- */
size_t rsc_pca_transform_workspace_bytes(int32_t n_cols, int32_t n_comps);
int rsc_pca_transform(const rsc_csr* X, const double* V, const double* gene_mean, int32_t n_comps,
                      float* out, void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_hvg_select_cell_ranger: cell-ranger-flavour HVG selection
 * (reading R18) from the mean / variance of the NORMALISED, non-logged
 * matrix (mean_lin / var_lin of rsc_normalize_log1p_moments):
 *   mean == 0 -> 1e-12; d = var / mean; bins = the intervals (e_k, e_{k+1}] of the edges -inf, P10,
 *   P15, .., P100 of the means (linear interpolation; equal edges merged), +inf;
 *   z = (d - median_bin(d)) / (median_bin |d - median_bin(d)| / 0.6745)  (IEEE: a zero MAD gives
 *   +-inf or NaN); cutoff = n_top-th largest non-NaN z; mask = z >= cutoff.
 *   Outputs as rsc_hvg_select (out_disp, out_disp_norm, out_bin, out_indices optional).
 *   1 <= n_genes <= 65 535, n_top >= 1.
 *
 * rsc_hvg_merge_batches: per-batch HVG (reading R19): the selection was run once per batch of cells
 * (row ranges of the matrix; any flavour); masks uint8[n_batches][n_genes] and disp_norm
 * double[n_batches][n_genes] hold its per-batch outputs.  Per gene: out_nbatches = number of
 * batches that selected it, out_disp_norm_mean = mean of its non-NaN normalised dispersions (NaN
 * if none); genes are ranked by (nbatches, mean dispersion) descending, NaN last inside a level,
 * and every gene at or above the n_top-th is selected.  1 <= n_batches <= 256.
 * ------------------------------------------------------------------------------- */
size_t rsc_hvg_select_cell_ranger_workspace_bytes(int32_t n_genes);
int rsc_hvg_select_cell_ranger(int32_t n_genes, const double* gene_mean, const double* gene_var,
                               int32_t n_top, double* out_disp, double* out_disp_norm,
                               int32_t* out_bin, uint8_t* out_mask, int32_t* out_indices,
                               int32_t* out_count, void* ws, size_t ws_bytes, void* stream);
int rsc_hvg_merge_batches(int32_t n_genes, int32_t n_batches, const uint8_t* masks,
                          const double* disp_norm, int32_t n_top, int32_t* out_nbatches,
                          double* out_disp_norm_mean, uint8_t* out_mask, int32_t* out_indices,
                          int32_t* out_count, void* stream);

/* ---------------------------------------------------------------------------------
 * SURVEY.md 8(f) NEXT-3 (first half) -- rsc_scale_dense: z-score per gene with optional clip
 * ("scaling"), written as a DENSE row-major float32 [n_rows, n_cols] matrix
 * (run it after subsetting to the HVGs: the output has n_rows * n_cols elements):
 *     out[i][j] = clip((x_ij - gene_mean[j]) / sd_j),  sd_j = sqrt(gene_var[j]), 1 where it is 0
 *   zero_center = 0: out = x_ij / sd_j (zeros stay zero).  max_value > 0: clip to
 *   [-max_value, max_value] (zero_center) or (-inf, max_value]; max_value <= 0: no clip.
 *   gene_mean / gene_var: e.g. mean_log / var_log of rsc_normalize_log1p_moments (ddof 1).
 *   ws: rsc_scale_dense_workspace_bytes(n_cols) bytes.  X is not modified.
 * ------------------------------------------------------------------------------- */
size_t rsc_scale_dense_workspace_bytes(int32_t n_cols);
int rsc_scale_dense(const rsc_csr* X, const double* gene_mean, const double* gene_var,
                    float max_value, int zero_center, float* out, void* ws, size_t ws_bytes,
                    void* stream);

/* ---------------------------------------------------------------------------------
 * SURVEY.md 8(f) NEXT-3 (second half) -- rsc_gram_cov: the sparse PCA front end of PAPER.md:L95
 * ("Principal component analysis"; L137 "centered Gram matrix construction") for X in R^{n x p}
 * (run it on the HVG-subset, log-normalised matrix):
 *     out_mean[j]    mu = (1/n) X^T 1                                  double[p]
 *     out_gram[a][b] S  = X^T X (upper triangle accumulated, mirrored) double[p * p], row-major
 *     out_cov[a][b]  C  = (S - n mu mu^T) / (n - 1)  (implicit centring) double[p * p]
 *   Any output may be NULL.  The contraction runs on the tensor cores (tcgen05, fp32 accumulators
 *   in TMEM) on fp16 pairs hi + lo of x * 2^k (2^k chosen on the device from max |x|; 22
 *   significand bits), S = hi^T hi + hi^T lo + lo^T hi: fp32-equivalent accuracy, |S - S_exact| <=
 *   1e-5 |S_exact| entry-wise for non-negative data (DESIGN.md section 6 gives the budget); C is
 *   formed from S and the exact mu in double, so its error is that of S divided by n - 1.
 *   The result is bit-reproducible (no atomics).  n_rows >= 2, 1 <= n_cols <= 8192, |x| finite;
 *   rows need not be sorted.  ws: rsc_gram_cov_workspace_bytes(n_rows, n_cols, nnz) bytes (two
 *   dense fp16 planes of at most 262 144 rows, the partial tiles; <= 2 x 4.3 GB + 0.6 GB).
 * ------------------------------------------------------------------------------- */
size_t rsc_gram_cov_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);
int rsc_gram_cov(const rsc_csr* X, double* out_mean, double* out_gram, double* out_cov,
                 void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_hvg_select — Seurat-flavour highly-variable-gene selection on the device
 * ("based on per-gene mean and variance"; L39 "gene selection" kernel
 * that avoids CPU<->GPU transfers; L87 "follow the algorithmic implementations of
 * scanpy"; steps H1..H7 of DESIGN.md §3):
 *   mean==0 -> 1e-12; d = var/mean; [flags bit0] d==0 -> NaN, d = ln d, m = log1p(mean);
 *   n_bins equal-width right-closed bins over m (first edge lowered by 0.1 % of the
 *   range); z = (d - mean_bin(d)) / sd_bin(d) (ddof 1, NaNs skipped; a bin with one
 *   valid gene gives z = 1); cutoff = n_top-th largest non-NaN z; mask = z >= cutoff.
 *   Outputs (all optional except out_mask / out_count):
 *     out_mean_t, out_disp, out_disp_norm  double[n_genes]   m, d, z
 *     out_bin      int32[n_genes]
 *     out_mask     uint8[n_genes]          1 = selected
 *     out_indices  int32[n_genes]          selected genes, ascending; tail untouched
 *     out_count    int32[1]                number selected (>= n_top on ties; the number
 *                                          of non-NaN genes if that is smaller)
 *   1 <= n_bins <= 4096, n_top >= 1, n_genes >= 1.
 * ------------------------------------------------------------------------------- */
#define RSC_HVG_SEURAT_LOG 1
size_t rsc_hvg_select_workspace_bytes(int32_t n_genes, int32_t n_bins);
int rsc_hvg_select(int32_t n_genes, const double* gene_mean, const double* gene_var,
                   int32_t n_top, int32_t n_bins, int flags,
                   double* out_mean_t, double* out_disp, double* out_disp_norm,
                   int32_t* out_bin, uint8_t* out_mask, int32_t* out_indices,
                   int32_t* out_count, void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_hvg_select_no_alloc — rsc_hvg_select without a workspace argument, for callers that can
 * neither allocate device memory nor hand one in (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc).  Same operation, same kernels, same arguments and
 * outputs as rsc_hvg_select; the kernels' scratch lives in a device array
 * built into the library:
 *   * at most RSC_HVG_NO_ALLOC_MAX_GENES genes (2 MiB of device memory, held by every GPU
 *     that loads the library until the process exits); more genes -> RSC_ERR_INVALID_ARG,
 *     nothing is launched (use rsc_hvg_select with your own workspace);
 *   * the call allocates and frees nothing (no cudaMalloc / cudaFree, no allocating library
 *     routine); the first call on a device looks the array's address up once;
 *   * all calls on one device share the array: calls that OVERLAP on the GPU (different
 *     streams, concurrent graph replays) race on it and must be serialised by the caller.
 *     Nothing in it carries over between calls (every element is written before it is read).
 * rsc_hvg_select_no_alloc_max_genes() returns the limit the library was built with.
 * ------------------------------------------------------------------------------- */
#define RSC_HVG_NO_ALLOC_MAX_GENES 65536
int32_t rsc_hvg_select_no_alloc_max_genes(void);
int rsc_hvg_select_no_alloc(int32_t n_genes, const double* gene_mean, const double* gene_var,
                            int32_t n_top, int32_t n_bins, int flags,
                            double* out_mean_t, double* out_disp, double* out_disp_norm,
                            int32_t* out_bin, uint8_t* out_mask, int32_t* out_indices,
                            int32_t* out_count, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_preprocess — the whole chain in one call on device-resident data:
 * rsc_qc_metrics -> rsc_normalize_log1p_moments -> rsc_hvg_select (fed with the
 * linear-scale moments when hvg_on_linear != 0, else the log-scale ones; DESIGN.md
 * reading R8).  `out` collects the device output pointers; see rsc_outputs.
 * PRECONDITION (as rsc_qc_metrics): X->data holds integer counts.  The chain normalises with the
 * QC totals, which truncate every value to an integer before summing (reading R4); for
 * non-integer input (ambient-corrected or already normalised values) the row sums of x' then
 * differ from target_sum and nothing reports it -- call rsc_normalize_total with a NULL total
 * (float row sums), rsc_log1p and rsc_gene_moments instead.
 * ------------------------------------------------------------------------------- */
typedef struct {
  /* per cell [n_rows] */
  int64_t* cell_total_i64; float* cell_total_f32; int32_t* cell_n_genes;
  int64_t* cell_flag_total_i64; float* cell_flag_pct;
  /* per gene [n_cols] */
  int32_t* gene_n_cells; int64_t* gene_total_i64;
  double* mean_log; double* var_log; double* mean_lin; double* var_lin;
  double* hvg_mean_t; double* hvg_disp; double* hvg_disp_norm; int32_t* hvg_bin;
  uint8_t* hvg_mask; int32_t* hvg_indices;
  int32_t* hvg_count; /* [1] */
} rsc_outputs;

typedef struct {
  float target_sum;
  int32_t n_top;
  int32_t n_bins;
  int32_t ddof;
  int32_t which_moments;  /* RSC_MOMENTS_* bits                                */
  int32_t hvg_on_linear;  /* 1: HVG consumes linear-scale moments, 0: log-scale */
  int32_t hvg_flags;      /* RSC_HVG_* bits                                     */
} rsc_params;

size_t rsc_preprocess_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz, int32_t n_bins);
int rsc_preprocess(rsc_csr* X, const uint8_t* gene_flags, const rsc_params* prm,
                   const rsc_outputs* out, void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------
 * rsc_preprocess_host — the same chain for a matrix that lives in HOST memory
 * ("a single function transfers data to GPU memory").  `host_X` holds
 * HOST pointers (pinned memory recommended), `host_out` HOST output pointers (any may
 * be NULL); `host_data_out` optionally receives the log-normalised values.  The call
 * stages everything through the caller's device workspace `dev_ws` (size from
 * rsc_preprocess_host_workspace_bytes) and returns without synchronising; the caller
 * synchronises `stream` before reading the host outputs.  The matrix travels in row chunks: the
 * kernels of chunk k run on `stream` while chunk k + 1 is copied in and the x'' of chunk k - 1 is
 * copied out on two copy streams the library keeps per host thread and device (they start after
 * the work already queued on `stream`, and `stream` waits for them before the call's last
 * copies); the per-gene results of the chunks are added in chunk order.  Pinned host memory is
 * needed for the copies to overlap.
 * ------------------------------------------------------------------------------- */
size_t rsc_preprocess_host_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz, int32_t n_bins);
int rsc_preprocess_host(const rsc_csr* host_X, const uint8_t* host_gene_flags,
                        const rsc_params* prm, const rsc_outputs* host_out,
                        float* host_data_out, void* dev_ws, size_t dev_ws_bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* RSC_H_ */
