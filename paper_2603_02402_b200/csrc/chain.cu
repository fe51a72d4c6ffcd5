// Whole-chain entry points: rsc_preprocess (device-resident matrix) and rsc_preprocess_host
// (host matrix staged through a caller-provided device workspace).  PAPER.md:L47 / L145
// workflow order, L31 "a single function transfers data to GPU memory".
#include <math.h>

#include "common.cuh"

namespace rsc {

struct Carver {
  unsigned char* base;
  size_t off = 0;
  explicit Carver(void* p) : base(static_cast<unsigned char*>(p)) {}
  template <typename T>
  T* take(size_t count) {
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += align_up(sizeof(T) * count, 256);
    return p;
  }
  void* take_bytes(size_t bytes) {
    void* p = base ? base + off : nullptr;
    off += align_up(bytes, 256);
    return p;
  }
};

struct ChainWs {
  int64_t* cell_total;
  int32_t* gene_n_cells;
  uint32_t* splits;
  double *mean_log, *var_log, *mean_lin, *var_lin;
  void *qc_ws, *fused_ws, *hvg_ws;
  size_t qc_bytes, fused_bytes, hvg_bytes;
  size_t total;
};

static ChainWs carve_chain(void* ws, int64_t n, int32_t G, int64_t nnz, int32_t n_bins) {
  Carver c(ws);
  ChainWs w;
  w.cell_total = c.take<int64_t>((size_t)n);
  w.gene_n_cells = c.take<int32_t>((size_t)G);
  w.splits = c.take<uint32_t>(rsc_row_splits_count(n, G));
  w.mean_log = c.take<double>((size_t)G);
  w.var_log = c.take<double>((size_t)G);
  w.mean_lin = c.take<double>((size_t)G);
  w.var_lin = c.take<double>((size_t)G);
  w.qc_bytes = qc_workspace_bytes(n, G, nnz);
  w.fused_bytes = fused_workspace_bytes(n, G, nnz);
  w.hvg_bytes = hvg_workspace_bytes(G, n_bins);
  w.qc_ws = c.take_bytes(w.qc_bytes);
  w.fused_ws = c.take_bytes(w.fused_bytes);
  w.hvg_ws = c.take_bytes(w.hvg_bytes);
  w.total = c.off;
  return w;
}

static int check_params(const rsc_params* p, const char* who) {
  RSC_CHECK_ARG(p != nullptr, "%s: params is NULL", who);
  RSC_CHECK_ARG(isfinite(p->target_sum) && p->target_sum > 0.0f, "%s: target_sum must be > 0", who);
  RSC_CHECK_ARG(p->n_top >= 1, "%s: n_top < 1", who);
  RSC_CHECK_ARG(p->n_bins >= 1 && p->n_bins <= 4096, "%s: n_bins must be in [1, 4096]", who);
  RSC_CHECK_ARG(p->ddof == 0 || p->ddof == 1, "%s: ddof must be 0 or 1", who);
  RSC_CHECK_ARG((p->which_moments & 3) != 0 && (p->which_moments & ~7) == 0,
                "%s: which_moments must request RSC_MOMENTS_LOG and / or RSC_MOMENTS_LIN", who);
  RSC_CHECK_ARG(p->hvg_on_linear ? (p->which_moments & RSC_MOMENTS_LIN)
                                 : (p->which_moments & RSC_MOMENTS_LOG),
                "%s: which_moments does not produce the moments HVG is asked to consume", who);
  return RSC_OK;
}

static int run_chain(rsc_csr* X, const uint8_t* gene_flags, const rsc_params* prm,
                     const rsc_outputs* out, void* ws, cudaStream_t st) {
  ChainWs w = carve_chain(ws, X->n_rows, X->n_cols, X->nnz, prm->n_bins);
  int64_t* cell_total = out->cell_total_i64 ? out->cell_total_i64 : w.cell_total;
  int32_t* gene_n_cells = out->gene_n_cells ? out->gene_n_cells : w.gene_n_cells;
  double* mean_log = out->mean_log ? out->mean_log : w.mean_log;
  double* var_log = out->var_log ? out->var_log : w.var_log;
  double* mean_lin = out->mean_lin ? out->mean_lin : w.mean_lin;
  double* var_lin = out->var_lin ? out->var_lin : w.var_lin;

  uint32_t* splits = (X->flags & RSC_CSR_SORTED) ? w.splits : nullptr;
  // only the split entries the fused pass will read (its group edges) are produced
  int32_t need[32];
  int32_t n_need = fused_split_blocks(X->n_cols, prm->which_moments, need, 32);
  if (n_need > 32) n_need = 0;
  int rc = launch_qc(*X, gene_flags, cell_total, out->cell_total_f32, out->cell_n_genes,
                     out->cell_flag_total_i64, out->cell_flag_pct, gene_n_cells,
                     out->gene_total_i64, splits, need, n_need, w.qc_ws, w.qc_bytes, st);
  if (rc) return rc;
  rc = launch_fused(*X, prm->target_sum, cell_total, gene_n_cells, splits, prm->which_moments, prm->ddof,
                    mean_log, var_log, mean_lin, var_lin, nullptr, w.fused_ws, w.fused_bytes, st);
  if (rc) return rc;
  const double* hm = prm->hvg_on_linear ? mean_lin : mean_log;
  const double* hv = prm->hvg_on_linear ? var_lin : var_log;
  return launch_hvg(X->n_cols, hm, hv, prm->n_top, prm->n_bins, prm->hvg_flags, out->hvg_mean_t,
                    out->hvg_disp, out->hvg_disp_norm, out->hvg_bin, out->hvg_mask,
                    out->hvg_indices, out->hvg_count, w.hvg_ws, w.hvg_bytes, st);
}

struct HostWs {
  int64_t* indptr; int32_t* indices; float* data; uint8_t* flags;
  rsc_outputs o;
  void* chain_ws; size_t chain_bytes;
  size_t total;
};

static HostWs carve_host(void* ws, int64_t n, int32_t G, int64_t nnz, int32_t n_bins) {
  Carver c(ws);
  HostWs h;
  h.indptr = c.take<int64_t>((size_t)n + 1);
  h.indices = c.take<int32_t>((size_t)nnz);
  h.data = c.take<float>((size_t)nnz);
  h.flags = c.take<uint8_t>((size_t)G);
  h.o.cell_total_i64 = c.take<int64_t>((size_t)n);
  h.o.cell_total_f32 = c.take<float>((size_t)n);
  h.o.cell_n_genes = c.take<int32_t>((size_t)n);
  h.o.cell_flag_total_i64 = c.take<int64_t>((size_t)n);
  h.o.cell_flag_pct = c.take<float>((size_t)n);
  h.o.gene_n_cells = c.take<int32_t>((size_t)G);
  h.o.gene_total_i64 = c.take<int64_t>((size_t)G);
  h.o.mean_log = c.take<double>((size_t)G);
  h.o.var_log = c.take<double>((size_t)G);
  h.o.mean_lin = c.take<double>((size_t)G);
  h.o.var_lin = c.take<double>((size_t)G);
  h.o.hvg_mean_t = c.take<double>((size_t)G);
  h.o.hvg_disp = c.take<double>((size_t)G);
  h.o.hvg_disp_norm = c.take<double>((size_t)G);
  h.o.hvg_bin = c.take<int32_t>((size_t)G);
  h.o.hvg_mask = c.take<uint8_t>((size_t)G);
  h.o.hvg_indices = c.take<int32_t>((size_t)G);
  h.o.hvg_count = c.take<int32_t>(1);
  h.chain_bytes = carve_chain(nullptr, n, G, nnz, n_bins).total;
  h.chain_ws = c.take_bytes(h.chain_bytes);
  h.total = c.off;
  return h;
}

template <typename T>
static int d2h(T* host, const T* dev, size_t count, cudaStream_t st) {
  if (host == nullptr || count == 0) return RSC_OK;
  RSC_CUDA(cudaMemcpyAsync(host, dev, sizeof(T) * count, cudaMemcpyDeviceToHost, st));
  return RSC_OK;
}

}  // namespace rsc

using namespace rsc;

extern "C" {

size_t rsc_preprocess_workspace_bytes(int64_t n, int32_t G, int64_t nnz, int32_t n_bins) {
  return carve_chain(nullptr, n, G, nnz, n_bins).total;
}

int rsc_preprocess(rsc_csr* X, const uint8_t* gene_flags, const rsc_params* prm,
                   const rsc_outputs* out, void* ws, size_t ws_bytes, void* stream) {
  RSC_CHECK_ARG(X != nullptr && out != nullptr, "rsc_preprocess: X / out is NULL");
  RSC_CHECK_ARG(X->n_rows >= 0 && X->n_cols > 0 && X->nnz >= 0 && X->indptr != nullptr,
                "rsc_preprocess: bad CSR header");
  RSC_CHECK_ARG(X->nnz == 0 || (X->indices && X->data), "rsc_preprocess: indices / data is NULL");
  int rc = check_params(prm, "rsc_preprocess");
  if (rc) return rc;
  RSC_CHECK_ARG(X->n_rows - prm->ddof > 0, "rsc_preprocess: n_rows - ddof must be > 0");
  RSC_CHECK_ARG(out->hvg_mask && out->hvg_count, "rsc_preprocess: hvg_mask / hvg_count are required");
  if ((rc = check_device())) return rc;
  const size_t need = rsc_preprocess_workspace_bytes(X->n_rows, X->n_cols, X->nnz, prm->n_bins);
  if (ws == nullptr || ws_bytes < need || (reinterpret_cast<uintptr_t>(ws) & 255)) {
    set_error("rsc_preprocess: workspace too small or misaligned (have %zu, need %zu)", ws_bytes, need);
    return RSC_ERR_WORKSPACE;
  }
  return run_chain(X, gene_flags, prm, out, ws, static_cast<cudaStream_t>(stream));
}

size_t rsc_preprocess_host_workspace_bytes(int64_t n, int32_t G, int64_t nnz, int32_t n_bins) {
  return carve_host(nullptr, n, G, nnz, n_bins).total;
}

int rsc_preprocess_host(const rsc_csr* hX, const uint8_t* host_gene_flags, const rsc_params* prm,
                        const rsc_outputs* ho, float* host_data_out, void* dev_ws,
                        size_t dev_ws_bytes, void* stream) {
  RSC_CHECK_ARG(hX != nullptr && ho != nullptr, "rsc_preprocess_host: host_X / host_out is NULL");
  RSC_CHECK_ARG(hX->n_rows >= 0 && hX->n_cols > 0 && hX->nnz >= 0 && hX->indptr != nullptr,
                "rsc_preprocess_host: bad CSR header");
  RSC_CHECK_ARG(hX->nnz == 0 || (hX->indices && hX->data), "rsc_preprocess_host: indices / data is NULL");
  int rc = check_params(prm, "rsc_preprocess_host");
  if (rc) return rc;
  RSC_CHECK_ARG(hX->n_rows - prm->ddof > 0, "rsc_preprocess_host: n_rows - ddof must be > 0");
  if ((rc = check_device())) return rc;
  const int64_t n = hX->n_rows, nnz = hX->nnz;
  const int32_t G = hX->n_cols;
  HostWs h = carve_host(dev_ws, n, G, nnz, prm->n_bins);
  if (dev_ws == nullptr || dev_ws_bytes < h.total || (reinterpret_cast<uintptr_t>(dev_ws) & 255)) {
    set_error("rsc_preprocess_host: workspace too small or misaligned (have %zu, need %zu)",
              dev_ws_bytes, h.total);
    return RSC_ERR_WORKSPACE;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  RSC_CUDA(cudaMemcpyAsync(h.indptr, hX->indptr, sizeof(int64_t) * (size_t)(n + 1), cudaMemcpyHostToDevice, st));
  if (nnz) {
    RSC_CUDA(cudaMemcpyAsync(h.indices, hX->indices, sizeof(int32_t) * (size_t)nnz, cudaMemcpyHostToDevice, st));
    RSC_CUDA(cudaMemcpyAsync(h.data, hX->data, sizeof(float) * (size_t)nnz, cudaMemcpyHostToDevice, st));
  }
  const uint8_t* dflags = nullptr;
  if (host_gene_flags) {
    RSC_CUDA(cudaMemcpyAsync(h.flags, host_gene_flags, (size_t)G, cudaMemcpyHostToDevice, st));
    dflags = h.flags;
  }
  rsc_csr dX = *hX;
  dX.indptr = h.indptr; dX.indices = h.indices; dX.data = h.data;
  if ((rc = run_chain(&dX, dflags, prm, &h.o, h.chain_ws, st))) return rc;
  const size_t sn = (size_t)n, sg = (size_t)G;
  if ((rc = d2h(ho->cell_total_i64, h.o.cell_total_i64, sn, st))) return rc;
  if ((rc = d2h(ho->cell_total_f32, h.o.cell_total_f32, sn, st))) return rc;
  if ((rc = d2h(ho->cell_n_genes, h.o.cell_n_genes, sn, st))) return rc;
  if ((rc = d2h(ho->cell_flag_total_i64, h.o.cell_flag_total_i64, sn, st))) return rc;
  if ((rc = d2h(ho->cell_flag_pct, h.o.cell_flag_pct, sn, st))) return rc;
  if ((rc = d2h(ho->gene_n_cells, h.o.gene_n_cells, sg, st))) return rc;
  if ((rc = d2h(ho->gene_total_i64, h.o.gene_total_i64, sg, st))) return rc;
  if (prm->which_moments & RSC_MOMENTS_LOG) {
    if ((rc = d2h(ho->mean_log, h.o.mean_log, sg, st))) return rc;
    if ((rc = d2h(ho->var_log, h.o.var_log, sg, st))) return rc;
  }
  if (prm->which_moments & RSC_MOMENTS_LIN) {
    if ((rc = d2h(ho->mean_lin, h.o.mean_lin, sg, st))) return rc;
    if ((rc = d2h(ho->var_lin, h.o.var_lin, sg, st))) return rc;
  }
  if ((rc = d2h(ho->hvg_mean_t, h.o.hvg_mean_t, sg, st))) return rc;
  if ((rc = d2h(ho->hvg_disp, h.o.hvg_disp, sg, st))) return rc;
  if ((rc = d2h(ho->hvg_disp_norm, h.o.hvg_disp_norm, sg, st))) return rc;
  if ((rc = d2h(ho->hvg_bin, h.o.hvg_bin, sg, st))) return rc;
  if ((rc = d2h(ho->hvg_mask, h.o.hvg_mask, sg, st))) return rc;
  if ((rc = d2h(ho->hvg_indices, h.o.hvg_indices, sg, st))) return rc;
  if ((rc = d2h(ho->hvg_count, h.o.hvg_count, 1, st))) return rc;
  if (host_data_out && nnz) {
    RSC_CUDA(cudaMemcpyAsync(host_data_out, h.data, sizeof(float) * (size_t)nnz, cudaMemcpyDeviceToHost, st));
  }
  return RSC_OK;
}

}  // extern "C"
