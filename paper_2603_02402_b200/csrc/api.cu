// C ABI of librsc_b200 (include/rsc.h): host-side argument validation, workspace carving,
// dispatch between the sorted-row shared-memory kernels and the generic L2-atomic kernels,
// and the two whole-chain entry points.  No device allocation, no stream synchronisation.
#include <math.h>
#include <stdarg.h>
#include <string.h>

#include "common.cuh"

namespace rsc {

static thread_local char g_err[512] = "";
std::atomic<unsigned long long> g_launch_count{0};
Options g_opt;

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

// per host thread (the current device is a per-thread notion): no shared mutable state
static thread_local int g_dev_checked = -1;   // device ordinal whose capability was verified
static thread_local int g_sm_count = kNumSMs;

int check_device() {
  int dev = -1;
  RSC_CUDA(cudaGetDevice(&dev));
  if (dev == g_dev_checked) return RSC_OK;
  int major = 0, sms = 0;
  RSC_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  RSC_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (major != 10) {
    set_error("device %d has compute capability %d.x; librsc_b200 is built for sm_100a only", dev,
              major);
    return RSC_ERR_UNSUPPORTED;
  }
  g_sm_count = sms;
  g_dev_checked = dev;
  return RSC_OK;
}

int sm_count() { return g_sm_count; }

static int check_csr(const rsc_csr* X, const char* who, bool need_data) {
  RSC_CHECK_ARG(X != nullptr, "%s: X is NULL", who);
  RSC_CHECK_ARG(X->n_rows >= 0, "%s: n_rows < 0", who);
  RSC_CHECK_ARG(X->n_cols > 0, "%s: n_cols <= 0", who);
  RSC_CHECK_ARG(X->nnz >= 0, "%s: nnz < 0", who);
  RSC_CHECK_ARG(X->indptr != nullptr, "%s: indptr is NULL", who);
  RSC_CHECK_ARG(X->nnz == 0 || X->indices != nullptr, "%s: indices is NULL", who);
  RSC_CHECK_ARG(X->nnz == 0 || !need_data || X->data != nullptr, "%s: data is NULL", who);
  return RSC_OK;
}

static int check_ws(const char* who, void* ws, size_t have, size_t need) {
  if (need == 0) return RSC_OK;
  if (ws == nullptr || have < need || (reinterpret_cast<uintptr_t>(ws) & 255)) {
    set_error("%s: workspace too small or misaligned (have %zu, need %zu, 256-byte aligned)", who,
              have, need);
    return RSC_ERR_WORKSPACE;
  }
  return RSC_OK;
}

// implemented in generic.cu
int launch_moments_generic(const rsc_csr&, int, double*, double*, cudaStream_t);
int finalize_moments(int32_t, int64_t, int, const double*, const double*, double*, double*,
                     cudaStream_t);

// implemented in fused.cu: the moments-only pass on the streaming skeleton
size_t moments_fast_workspace_bytes(int64_t n_rows, int32_t n_cols);
bool moments_fast_ok(const rsc_csr& X);
int launch_moments_fast(const rsc_csr& X, int ddof, double* mean, double* var, double* sum, double* sumsq,
                        void* ws, cudaStream_t st);

size_t moments_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t) {
  return moments_fast_workspace_bytes(n_rows, n_cols);
}

int launch_moments(const rsc_csr& X, int transform, int ddof, double* mean, double* var,
                   double* sum, double* sumsq, void* ws, size_t, cudaStream_t st) {
  const size_t gsz = align_up(sizeof(double) * (size_t)X.n_cols, 256);
  unsigned char* w = static_cast<unsigned char*>(ws);
  // transform 0 on sorted rows: on-chip integer accumulators; expm1 needs fp64 values (1e-9 bar),
  // which only the generic L2-atomic kernel provides
  if (transform == 0 && moments_fast_ok(X)) return launch_moments_fast(X, ddof, mean, var, sum, sumsq, ws, st);
  double* S1 = sum ? sum : reinterpret_cast<double*>(w);
  double* S2 = sumsq ? sumsq : reinterpret_cast<double*>(w + gsz);
  int rc = launch_moments_generic(X, transform, S1, S2, st);
  if (rc != RSC_OK) return rc;
  return finalize_moments(X.n_cols, X.n_rows, ddof, S1, S2, mean, var, st);
}

}  // namespace rsc

using namespace rsc;

extern "C" {

const char* rsc_last_error(void) { return g_err; }
const char* rsc_version(void) { return "0.1.0"; }
uint64_t rsc_kernel_launch_count(void) { return g_launch_count.load(std::memory_order_relaxed); }

int rsc_set_option(const char* key, long long value) {
  RSC_CHECK_ARG(key != nullptr, "rsc_set_option: key is NULL");
  if (!strcmp(key, "fused_row_budget")) {
    RSC_CHECK_ARG(value >= 1 && value <= 256, "rsc_set_option: fused_row_budget must be in [1, 256]");
    g_opt.fused_row_budget = (int)value;
  } else if (!strcmp(key, "flush_all")) {
    g_opt.flush_all = value != 0;
  } else if (!strcmp(key, "qc_row_budget")) {
    RSC_CHECK_ARG(value >= 1 && value <= 512, "rsc_set_option: qc_row_budget must be in [1, 512]");
    g_opt.qc_row_budget = (int)value;
  } else if (!strcmp(key, "grid_ctas")) {
    RSC_CHECK_ARG(value >= 0 && value <= 65535, "rsc_set_option: grid_ctas must be in [0, 65535]");
    g_opt.grid_ctas = (int)value;
  } else if (!strcmp(key, "force_generic")) {
    g_opt.force_generic = value != 0;
  } else if (!strcmp(key, "host_chunk_nnz")) {
    RSC_CHECK_ARG(value >= 0, "rsc_set_option: host_chunk_nnz must be >= 0");
    g_opt.host_chunk_nnz = value;
  } else if (!strcmp(key, "single_pass")) {
    g_opt.single_pass = value != 0;
  } else if (!strcmp(key, "hvg_single_cta")) {
    g_opt.hvg_single_cta = value != 0;
  } else {
    set_error("rsc_set_option: unknown key '%s'", key);
    return RSC_ERR_INVALID_ARG;
  }
  return RSC_OK;
}

size_t rsc_qc_metrics_workspace_bytes(int64_t n, int32_t G, int64_t nnz) {
  return qc_workspace_bytes(n, G, nnz);
}

size_t rsc_row_splits_count(int64_t n_rows, int32_t n_cols) {
  if (n_rows < 0 || n_cols <= 0) return 0;
  return (size_t)n_rows * ((size_t)split_blocks(n_cols) + 1);
}

int rsc_row_splits(const rsc_csr* X, uint32_t* row_splits, void* stream) {
  int rc = check_csr(X, "rsc_row_splits", false);
  if (rc) return rc;
  RSC_CHECK_ARG(row_splits != nullptr, "rsc_row_splits: row_splits is NULL");
  if ((rc = check_device())) return rc;
  return launch_row_splits(*X, row_splits, static_cast<cudaStream_t>(stream));
}

int rsc_qc_metrics_splits(const rsc_csr* X, const uint8_t* gene_flags, int64_t* cell_total_i64,
                          float* cell_total_f32, int32_t* cell_n_genes, int64_t* cell_flag_total_i64,
                          float* cell_flag_pct, int32_t* gene_n_cells, int64_t* gene_total_i64,
                          uint32_t* row_splits, const int32_t* split_blocks, int32_t n_split_blocks,
                          void* ws, size_t ws_bytes, void* stream) {
  int rc = check_csr(X, "rsc_qc_metrics", true);
  if (rc) return rc;
  RSC_CHECK_ARG(n_split_blocks >= 0 && n_split_blocks <= 32, "rsc_qc_metrics: n_split_blocks must be in [0, 32]");
  RSC_CHECK_ARG(n_split_blocks == 0 || split_blocks != nullptr, "rsc_qc_metrics: split_blocks is NULL");
  for (int i = 0; i < n_split_blocks; ++i)
    RSC_CHECK_ARG(split_blocks[i] >= 0 && split_blocks[i] <= ::rsc::split_blocks(X->n_cols),
                  "rsc_qc_metrics: split_blocks[%d] out of range", i);
  if ((rc = check_device())) return rc;
  if ((rc = check_ws("rsc_qc_metrics", ws, ws_bytes, qc_workspace_bytes(X->n_rows, X->n_cols, X->nnz))))
    return rc;
  if (!(X->flags & RSC_CSR_SORTED)) row_splits = nullptr;
  return launch_qc(*X, gene_flags, cell_total_i64, cell_total_f32, cell_n_genes,
                   cell_flag_total_i64, cell_flag_pct, gene_n_cells, gene_total_i64, row_splits,
                   split_blocks, n_split_blocks, ws, ws_bytes, static_cast<cudaStream_t>(stream));
}

int rsc_qc_metrics(const rsc_csr* X, const uint8_t* gene_flags, int64_t* cell_total_i64,
                   float* cell_total_f32, int32_t* cell_n_genes, int64_t* cell_flag_total_i64,
                   float* cell_flag_pct, int32_t* gene_n_cells, int64_t* gene_total_i64,
                   uint32_t* row_splits, void* ws, size_t ws_bytes, void* stream) {
  return rsc_qc_metrics_splits(X, gene_flags, cell_total_i64, cell_total_f32, cell_n_genes,
                               cell_flag_total_i64, cell_flag_pct, gene_n_cells, gene_total_i64,
                               row_splits, nullptr, 0, ws, ws_bytes, stream);
}

int32_t rsc_moments_split_blocks(int32_t n_cols, int which_moments, int32_t* blocks_out, int32_t cap) {
  if (n_cols <= 0 || blocks_out == nullptr || cap < 0) return 0;
  return fused_split_blocks(n_cols, which_moments, blocks_out, cap);
}

int rsc_normalize_total(rsc_csr* X, float target_sum, const int64_t* cell_total_i64,
                        float* cell_scale_out, void* stream) {
  int rc = check_csr(X, "rsc_normalize_total", true);
  if (rc) return rc;
  RSC_CHECK_ARG(isfinite(target_sum) && target_sum > 0.0f,
                "rsc_normalize_total: target_sum must be finite and > 0");
  if ((rc = check_device())) return rc;
  return launch_normalize(*X, target_sum, cell_total_i64, cell_scale_out,
                          static_cast<cudaStream_t>(stream));
}

int rsc_log1p(rsc_csr* X, void* stream) {
  int rc = check_csr(X, "rsc_log1p", true);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  return launch_log1p(*X, static_cast<cudaStream_t>(stream));
}

size_t rsc_gene_moments_workspace_bytes(int64_t n, int32_t G, int64_t nnz) {
  return moments_workspace_bytes(n, G, nnz);
}

int rsc_gene_moments(const rsc_csr* X, int transform, int ddof, double* gene_mean,
                     double* gene_var, double* gene_sum, double* gene_sumsq, void* ws,
                     size_t ws_bytes, void* stream) {
  int rc = check_csr(X, "rsc_gene_moments", true);
  if (rc) return rc;
  RSC_CHECK_ARG(transform == 0 || transform == 1, "rsc_gene_moments: transform must be 0 or 1");
  RSC_CHECK_ARG(ddof == 0 || ddof == 1, "rsc_gene_moments: ddof must be 0 or 1");
  RSC_CHECK_ARG(X->n_rows - ddof > 0, "rsc_gene_moments: n_rows - ddof must be > 0");
  RSC_CHECK_ARG(gene_mean != nullptr && gene_var != nullptr,
                "rsc_gene_moments: gene_mean / gene_var are required");
  if ((rc = check_device())) return rc;
  if ((rc = check_ws("rsc_gene_moments", ws, ws_bytes,
                     moments_workspace_bytes(X->n_rows, X->n_cols, X->nnz))))
    return rc;
  return launch_moments(*X, transform, ddof, gene_mean, gene_var, gene_sum, gene_sumsq, ws,
                        ws_bytes, static_cast<cudaStream_t>(stream));
}

size_t rsc_normalize_log1p_moments_workspace_bytes(int64_t n, int32_t G, int64_t nnz) {
  return fused_workspace_bytes(n, G, nnz);
}

int rsc_normalize_log1p_moments(rsc_csr* X, float target_sum, const int64_t* cell_total_i64,
                                const int32_t* gene_n_cells, const uint32_t* row_splits,
                                int which_moments, int ddof, double* mean_log, double* var_log, double* mean_lin,
                                double* var_lin, double* gene_sums_out, void* ws, size_t ws_bytes,
                                void* stream) {
  int rc = check_csr(X, "rsc_normalize_log1p_moments", true);
  if (rc) return rc;
  RSC_CHECK_ARG(isfinite(target_sum) && target_sum > 0.0f,
                "rsc_normalize_log1p_moments: target_sum must be finite and > 0");
  RSC_CHECK_ARG(cell_total_i64 != nullptr, "rsc_normalize_log1p_moments: cell_total_i64 is required");
  RSC_CHECK_ARG((which_moments & ~7) == 0, "rsc_normalize_log1p_moments: bad which_moments");
  RSC_CHECK_ARG(ddof == 0 || ddof == 1, "rsc_normalize_log1p_moments: ddof must be 0 or 1");
  RSC_CHECK_ARG((which_moments & 3) == 0 || X->n_rows - ddof > 0,
                "rsc_normalize_log1p_moments: n_rows - ddof must be > 0");
  RSC_CHECK_ARG(!(which_moments & RSC_MOMENTS_LOG) || (mean_log && var_log),
                "rsc_normalize_log1p_moments: mean_log / var_log required with RSC_MOMENTS_LOG");
  RSC_CHECK_ARG(!(which_moments & RSC_MOMENTS_LIN) || (mean_lin && var_lin),
                "rsc_normalize_log1p_moments: mean_lin / var_lin required with RSC_MOMENTS_LIN");
  if ((rc = check_device())) return rc;
  if ((rc = check_ws("rsc_normalize_log1p_moments", ws, ws_bytes,
                     fused_workspace_bytes(X->n_rows, X->n_cols, X->nnz))))
    return rc;
  return launch_fused(*X, target_sum, cell_total_i64, gene_n_cells, row_splits, which_moments, ddof,
                      mean_log, var_log, mean_lin, var_lin, gene_sums_out, ws, ws_bytes,
                      static_cast<cudaStream_t>(stream));
}

int rsc_moments_finalize(int32_t n_genes, int64_t n_rows_total, int ddof, const double* S1,
                         const double* S2, double* gene_mean, double* gene_var, void* stream) {
  RSC_CHECK_ARG(n_genes >= 1, "rsc_moments_finalize: n_genes < 1");
  RSC_CHECK_ARG(S1 && S2 && gene_mean && gene_var, "rsc_moments_finalize: NULL pointer");
  RSC_CHECK_ARG(ddof == 0 || ddof == 1, "rsc_moments_finalize: ddof must be 0 or 1");
  RSC_CHECK_ARG(n_rows_total - ddof > 0, "rsc_moments_finalize: n_rows_total - ddof must be > 0");
  int rc = check_device();
  if (rc) return rc;
  return finalize_moments(n_genes, n_rows_total, ddof, S1, S2, gene_mean, gene_var,
                          static_cast<cudaStream_t>(stream));
}

size_t rsc_hvg_select_workspace_bytes(int32_t G, int32_t n_bins) {
  return hvg_workspace_bytes(G, n_bins);
}

int rsc_filter_masks(int64_t n_rows, int32_t n_cols, const int32_t* cell_n_genes,
                     const int64_t* cell_total_i64, const float* cell_flag_pct,
                     const int32_t* gene_n_cells, const int64_t* gene_total_i64,
                     const rsc_filter_params* prm, uint8_t* cell_keep, uint8_t* gene_keep, void* stream) {
  RSC_CHECK_ARG(prm != nullptr, "rsc_filter_masks: params is NULL");
  RSC_CHECK_ARG(n_rows >= 0 && n_cols >= 0, "rsc_filter_masks: negative size");
  RSC_CHECK_ARG(!(prm->max_pct_flag != prm->max_pct_flag), "rsc_filter_masks: max_pct_flag is NaN");
  int rc = check_device();
  if (rc) return rc;
  return launch_filter_masks(n_rows, n_cols, cell_n_genes, cell_total_i64, cell_flag_pct, gene_n_cells,
                             gene_total_i64, *prm, cell_keep, gene_keep, static_cast<cudaStream_t>(stream));
}

size_t rsc_subset_csr_workspace_bytes(int64_t n_rows, int32_t n_cols) {
  return subset_workspace_bytes(n_rows, n_cols);
}

int rsc_subset_csr_plan(const rsc_csr* X, const uint8_t* keep_rows, const uint8_t* keep_cols,
                        int64_t* out_indptr, int64_t* out_counts, void* ws, size_t ws_bytes,
                        void* stream) {
  int rc = check_csr(X, "rsc_subset_csr_plan", false);
  if (rc) return rc;
  RSC_CHECK_ARG(out_indptr != nullptr && out_counts != nullptr, "rsc_subset_csr_plan: output is NULL");
  if ((rc = check_device())) return rc;
  if ((rc = check_ws("rsc_subset_csr_plan", ws, ws_bytes, subset_workspace_bytes(X->n_rows, X->n_cols))))
    return rc;
  return launch_subset_plan(*X, keep_rows, keep_cols, out_indptr, out_counts, ws,
                            static_cast<cudaStream_t>(stream));
}

int rsc_subset_csr_fill(const rsc_csr* X, const uint8_t* keep_rows, int32_t* out_indices,
                        float* out_data, void* ws, size_t ws_bytes, void* stream) {
  int rc = check_csr(X, "rsc_subset_csr_fill", true);
  if (rc) return rc;
  if ((rc = check_device())) return rc;
  if ((rc = check_ws("rsc_subset_csr_fill", ws, ws_bytes, subset_workspace_bytes(X->n_rows, X->n_cols))))
    return rc;
  return launch_subset_fill(*X, keep_rows, out_indices, out_data, ws, static_cast<cudaStream_t>(stream));
}

int rsc_hvg_cutoffs(int32_t n_genes, const double* mean_t, const double* disp_norm,
                    double min_mean, double max_mean, double min_disp, double max_disp,
                    uint8_t* out_mask, int32_t* out_indices, int32_t* out_count, void* stream) {
  RSC_CHECK_ARG(n_genes > 0, "rsc_hvg_cutoffs: n_genes <= 0");
  RSC_CHECK_ARG(mean_t != nullptr && disp_norm != nullptr, "rsc_hvg_cutoffs: input is NULL");
  RSC_CHECK_ARG(out_mask != nullptr && out_count != nullptr, "rsc_hvg_cutoffs: out_mask / out_count is NULL");
  RSC_CHECK_ARG(!(min_mean != min_mean) && !(max_mean != max_mean) && !(min_disp != min_disp) &&
                !(max_disp != max_disp), "rsc_hvg_cutoffs: a bound is NaN");
  int rc = check_device();
  if (rc) return rc;
  return launch_hvg_cutoffs(n_genes, mean_t, disp_norm, min_mean, max_mean, min_disp, max_disp, out_mask,
                            out_indices, out_count, static_cast<cudaStream_t>(stream));
}

size_t rsc_hvg_select_cell_ranger_workspace_bytes(int32_t n_genes) { return hvg_cell_ranger_workspace_bytes(n_genes); }

int rsc_hvg_select_cell_ranger(int32_t n_genes, const double* gene_mean, const double* gene_var, int32_t n_top,
                               double* out_disp, double* out_disp_norm, int32_t* out_bin, uint8_t* out_mask,
                               int32_t* out_indices, int32_t* out_count, void* ws, size_t ws_bytes, void* stream) {
  RSC_CHECK_ARG(n_genes >= 1 && n_genes <= 65535, "rsc_hvg_select_cell_ranger: n_genes must be in [1, 65535]");
  RSC_CHECK_ARG(gene_mean != nullptr && gene_var != nullptr, "rsc_hvg_select_cell_ranger: mean / var is NULL");
  RSC_CHECK_ARG(n_top >= 1, "rsc_hvg_select_cell_ranger: n_top < 1");
  RSC_CHECK_ARG(out_mask != nullptr && out_count != nullptr, "rsc_hvg_select_cell_ranger: out_mask / out_count is NULL");
  int rc = check_device();
  if (rc) return rc;
  if ((rc = check_ws("rsc_hvg_select_cell_ranger", ws, ws_bytes, hvg_cell_ranger_workspace_bytes(n_genes)))) return rc;
  return launch_hvg_cell_ranger(n_genes, gene_mean, gene_var, n_top, out_disp, out_disp_norm, out_bin, out_mask,
                                out_indices, out_count, ws, static_cast<cudaStream_t>(stream));
}

int rsc_hvg_merge_batches(int32_t n_genes, int32_t n_batches, const uint8_t* masks, const double* disp_norm,
                          int32_t n_top, int32_t* out_nbatches, double* out_disp_norm_mean, uint8_t* out_mask,
                          int32_t* out_indices, int32_t* out_count, void* stream) {
  RSC_CHECK_ARG(n_genes >= 1, "rsc_hvg_merge_batches: n_genes < 1");
  RSC_CHECK_ARG(n_batches >= 1 && n_batches <= 256, "rsc_hvg_merge_batches: n_batches must be in [1, 256]");
  RSC_CHECK_ARG(masks != nullptr && disp_norm != nullptr, "rsc_hvg_merge_batches: masks / disp_norm is NULL");
  RSC_CHECK_ARG(n_top >= 1, "rsc_hvg_merge_batches: n_top < 1");
  RSC_CHECK_ARG(out_nbatches != nullptr && out_disp_norm_mean != nullptr && out_mask != nullptr && out_count != nullptr,
                "rsc_hvg_merge_batches: a required output is NULL");
  int rc = check_device();
  if (rc) return rc;
  return launch_hvg_merge_batches(n_genes, n_batches, masks, disp_norm, n_top, out_nbatches, out_disp_norm_mean,
                                  out_mask, out_indices, out_count, static_cast<cudaStream_t>(stream));
}

size_t rsc_pca_transform_workspace_bytes(int32_t n_cols, int32_t n_comps) { return pca_workspace_bytes(n_cols, n_comps); }

int rsc_pca_transform(const rsc_csr* X, const double* V, const double* gene_mean, int32_t n_comps, float* out,
                      void* ws, size_t ws_bytes, void* stream) {
  int rc = check_csr(X, "rsc_pca_transform", true);
  if (rc) return rc;
  RSC_CHECK_ARG(pca_supported(n_comps), "rsc_pca_transform: n_comps must be in [1, 128]");
  RSC_CHECK_ARG(V != nullptr, "rsc_pca_transform: V is NULL");
  RSC_CHECK_ARG(out != nullptr || X->n_rows == 0, "rsc_pca_transform: out is NULL");
  if ((rc = check_device())) return rc;
  if ((rc = check_ws("rsc_pca_transform", ws, ws_bytes, pca_workspace_bytes(X->n_cols, n_comps)))) return rc;
  return launch_pca_transform(*X, V, gene_mean, n_comps, out, ws, static_cast<cudaStream_t>(stream));
}

size_t rsc_gram_cov_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz) {
  return gram_workspace_bytes(n_rows, n_cols, nnz);
}

int rsc_gram_cov(const rsc_csr* X, double* out_mean, double* out_gram, double* out_cov, void* ws,
                 size_t ws_bytes, void* stream) {
  int rc = check_csr(X, "rsc_gram_cov", true);
  if (rc) return rc;
  RSC_CHECK_ARG(X->n_rows >= 2, "rsc_gram_cov: needs at least two cells");
  RSC_CHECK_ARG(gram_supported(X->n_cols), "rsc_gram_cov: n_cols must be in [1, 8192]");
  if ((rc = check_device())) return rc;
  if ((rc = check_ws("rsc_gram_cov", ws, ws_bytes, gram_workspace_bytes(X->n_rows, X->n_cols, X->nnz)))) return rc;
  return launch_gram_cov(*X, out_mean, out_gram, out_cov, ws, ws_bytes, static_cast<cudaStream_t>(stream));
}

size_t rsc_scale_dense_workspace_bytes(int32_t n_cols) { return scale_workspace_bytes(n_cols); }

int rsc_scale_dense(const rsc_csr* X, const double* gene_mean, const double* gene_var,
                    float max_value, int zero_center, float* out, void* ws, size_t ws_bytes,
                    void* stream) {
  int rc = check_csr(X, "rsc_scale_dense", true);
  if (rc) return rc;
  RSC_CHECK_ARG(gene_mean != nullptr && gene_var != nullptr, "rsc_scale_dense: mean / var is NULL");
  RSC_CHECK_ARG(out != nullptr || X->n_rows == 0, "rsc_scale_dense: out is NULL");
  RSC_CHECK_ARG(!(max_value != max_value), "rsc_scale_dense: max_value is NaN");
  if ((rc = check_device())) return rc;
  if ((rc = check_ws("rsc_scale_dense", ws, ws_bytes, scale_workspace_bytes(X->n_cols)))) return rc;
  return launch_scale_dense(*X, gene_mean, gene_var, max_value, zero_center, out, ws,
                            static_cast<cudaStream_t>(stream));
}

int rsc_hvg_select(int32_t n_genes, const double* gene_mean, const double* gene_var, int32_t n_top,
                   int32_t n_bins, int flags, double* out_mean_t, double* out_disp,
                   double* out_disp_norm, int32_t* out_bin, uint8_t* out_mask,
                   int32_t* out_indices, int32_t* out_count, void* ws, size_t ws_bytes,
                   void* stream) {
  RSC_CHECK_ARG(n_genes >= 1, "rsc_hvg_select: n_genes < 1");
  RSC_CHECK_ARG(gene_mean && gene_var, "rsc_hvg_select: gene_mean / gene_var are required");
  RSC_CHECK_ARG(n_top >= 1, "rsc_hvg_select: n_top < 1");
  RSC_CHECK_ARG(n_bins >= 1 && n_bins <= 4096, "rsc_hvg_select: n_bins must be in [1, 4096]");
  RSC_CHECK_ARG(out_mask && out_count, "rsc_hvg_select: out_mask / out_count are required");
  int rc = check_device();
  if (rc) return rc;
  return launch_hvg(n_genes, gene_mean, gene_var, n_top, n_bins, flags, out_mean_t, out_disp,
                    out_disp_norm, out_bin, out_mask, out_indices, out_count, ws, ws_bytes,
                    static_cast<cudaStream_t>(stream));
}

}  // extern "C"
