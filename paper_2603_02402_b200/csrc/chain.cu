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

  if (single_pass_ok(*X, prm->which_moments) && !prm->hvg_on_linear &&
      single_workspace_bytes(X->n_rows, X->n_cols, X->nnz) <= w.fused_bytes) {
    // one pass over the matrix: QC + normalise + log1p + log-scale moments (single.cu)
    int rc1 = launch_single_pass(*X, gene_flags, prm->target_sum, prm->ddof, cell_total, out->cell_total_f32,
                                 out->cell_n_genes, out->cell_flag_total_i64, out->cell_flag_pct, gene_n_cells,
                                 out->gene_total_i64, mean_log, var_log, w.fused_ws, st);
    if (rc1) return rc1;
    return launch_hvg(X->n_cols, mean_log, var_log, prm->n_top, prm->n_bins, prm->hvg_flags, out->hvg_mean_t,
                      out->hvg_disp, out->hvg_disp_norm, out->hvg_bin, out->hvg_mask, out->hvg_indices,
                      out->hvg_count, w.hvg_ws, w.hvg_bytes, st);
  }
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
  // per-gene partial results of the row chunks (kHostMaxChunks each)
  int32_t* part_n_cells; int64_t* part_total; double* part_sums;   // [C][G], [C][G], [C][4 G]
  double* sums;                                                     // [4 G] added over the chunks
  size_t total;
};
constexpr int kHostMaxChunks = 16;

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
  h.part_n_cells = c.take<int32_t>((size_t)kHostMaxChunks * (size_t)G);
  h.part_total = c.take<int64_t>((size_t)kHostMaxChunks * (size_t)G);
  h.part_sums = c.take<double>((size_t)kHostMaxChunks * 4 * (size_t)G);
  h.sums = c.take<double>(4 * (size_t)G);
  h.total = c.off;
  return h;
}

// per-gene results of the row chunks added up (chunk order: a fixed summation order)
__global__ void __launch_bounds__(256)
host_chunk_reduce_kernel(int32_t G, int C, const int32_t* __restrict__ part_n_cells,
                         const int64_t* __restrict__ part_total, const double* __restrict__ part_sums,
                         int32_t* __restrict__ gene_n_cells, int64_t* __restrict__ gene_total,
                         double* __restrict__ sums) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= G) return;
  int32_t nc = 0;
  int64_t tt = 0;
  double s[4] = {0.0, 0.0, 0.0, 0.0};
  for (int c = 0; c < C; ++c) {
    nc += part_n_cells[(size_t)c * G + g];
    tt += part_total[(size_t)c * G + g];
#pragma unroll
    for (int k = 0; k < 4; ++k) s[k] += part_sums[((size_t)c * 4 + k) * G + g];
  }
  if (gene_n_cells) gene_n_cells[g] = nc;
  if (gene_total) gene_total[g] = tt;
#pragma unroll
  for (int k = 0; k < 4; ++k) sums[(size_t)k * G + g] = s[k];
}

// copy streams of the host entry point (one pair per host thread and device, created on first
// use and kept): the H2D copy of chunk k + 1 and the D2H copy of chunk k - 1 run beside the
// kernels of chunk k, which stay on the caller's stream
struct CopyStreams { int dev = -1; cudaStream_t in = nullptr, out = nullptr; };
static thread_local CopyStreams g_copy;
static int copy_streams(cudaStream_t* in, cudaStream_t* out) {
  int dev = -1;
  RSC_CUDA(cudaGetDevice(&dev));
  if (g_copy.dev != dev) {
    RSC_CUDA(cudaStreamCreateWithFlags(&g_copy.in, cudaStreamNonBlocking));
    RSC_CUDA(cudaStreamCreateWithFlags(&g_copy.out, cudaStreamNonBlocking));
    g_copy.dev = dev;
  }
  *in = g_copy.in; *out = g_copy.out;
  return RSC_OK;
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
  const uint8_t* dflags = nullptr;
  if (host_gene_flags) {
    RSC_CUDA(cudaMemcpyAsync(h.flags, host_gene_flags, (size_t)G, cudaMemcpyHostToDevice, st));
    dflags = h.flags;
  }
  // Row chunks of ~host_chunk_nnz stored entries (option; 150 M = 1.2 GB of H2D by default) (cut on the host from the host indptr).  The two
  // streaming passes need nothing beyond a chunk's own rows (the per-cell totals are row-local),
  // so chunk k is computed -- on the caller's stream -- while chunk k + 1 is copied in and the
  // x'' of chunk k - 1 is copied out on the two copy streams (PCIe is full duplex); the per-gene
  // results of the chunks are added up at the end, then moments, then HVG.
  const int64_t chunk_nnz = g_opt.host_chunk_nnz.load() > 0 ? (int64_t)g_opt.host_chunk_nnz.load() : nnz + 1;
  int64_t Cl = (nnz + chunk_nnz - 1) / chunk_nnz;
  int C = (int)(Cl > kHostMaxChunks ? kHostMaxChunks : Cl);
  C = C < 1 ? 1 : (C > kHostMaxChunks ? kHostMaxChunks : C);
  if (n < 4 * (int64_t)C) C = 1;
  int64_t rb[kHostMaxChunks + 1];
  rb[0] = 0;
  for (int c = 1; c < C; ++c) {                            // first row whose offset reaches c nnz / C
    const int64_t target = (int64_t)((double)nnz * c / C);
    int64_t lo = rb[c - 1], hi = n;
    while (lo < hi) {
      const int64_t mid = (lo + hi) >> 1;
      if (hX->indptr[mid] < target) lo = mid + 1; else hi = mid;
    }
    rb[c] = lo;
  }
  rb[C] = n;
  cudaStream_t s_in = st, s_out = st;
  cudaEvent_t ev_fork = nullptr, ev_in[kHostMaxChunks] = {}, ev_cmp[kHostMaxChunks] = {}, ev_out = nullptr;
  const bool piped = C > 1;
  if (piped) {
    if ((rc = copy_streams(&s_in, &s_out))) return rc;
    RSC_CUDA(cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming));
    RSC_CUDA(cudaEventCreateWithFlags(&ev_out, cudaEventDisableTiming));
    RSC_CUDA(cudaEventRecord(ev_fork, st));                // the copy streams start after the caller's earlier work
    RSC_CUDA(cudaStreamWaitEvent(s_in, ev_fork, 0));
    RSC_CUDA(cudaStreamWaitEvent(s_out, ev_fork, 0));
  }
  ChainWs w = carve_chain(h.chain_ws, n, G, nnz, prm->n_bins);
  const size_t K1 = (size_t)split_blocks(G) + 1;
  int32_t need[32];
  int32_t n_need = fused_split_blocks(G, prm->which_moments, need, 32);
  if (n_need > 32) n_need = 0;
  const bool sorted = (hX->flags & RSC_CSR_SORTED) != 0;
  for (int c = 0; c < C; ++c) {
    const int64_t r0 = rb[c], r1 = rb[c + 1];
    const int64_t p0 = hX->indptr[r0], p1 = hX->indptr[r1];
    if (p1 > p0) {
      RSC_CUDA(cudaMemcpyAsync(h.indices + p0, hX->indices + p0, sizeof(int32_t) * (size_t)(p1 - p0), cudaMemcpyHostToDevice, s_in));
      RSC_CUDA(cudaMemcpyAsync(h.data + p0, hX->data + p0, sizeof(float) * (size_t)(p1 - p0), cudaMemcpyHostToDevice, s_in));
    }
    if (piped) {
      RSC_CUDA(cudaEventCreateWithFlags(&ev_in[c], cudaEventDisableTiming));
      RSC_CUDA(cudaEventRecord(ev_in[c], s_in));
      RSC_CUDA(cudaStreamWaitEvent(st, ev_in[c], 0));
    }
    // the chunk as a CSR view: absolute offsets, so indices / data keep their base pointers
    rsc_csr Xc = *hX;
    Xc.n_rows = r1 - r0; Xc.indptr = h.indptr + r0; Xc.indices = h.indices; Xc.data = h.data;
    uint32_t* splits = sorted ? w.splits + (size_t)r0 * K1 : nullptr;
    int32_t* pn = h.part_n_cells + (size_t)c * G;
    int64_t* pt = h.part_total + (size_t)c * G;
    double* ps = h.part_sums + (size_t)c * 4 * G;
    RSC_CUDA(cudaMemsetAsync(ps, 0, sizeof(double) * 4 * (size_t)G, st));
    rc = launch_qc(Xc, dflags, h.o.cell_total_i64 + r0, h.o.cell_total_f32 + r0, h.o.cell_n_genes + r0,
                   h.o.cell_flag_total_i64 + r0, h.o.cell_flag_pct + r0, pn, pt, splits, need, n_need,
                   w.qc_ws, w.qc_bytes, st);
    if (rc) return rc;
    rc = launch_fused(Xc, prm->target_sum, h.o.cell_total_i64 + r0, pn, splits, prm->which_moments, prm->ddof,
                      w.mean_log, w.var_log, w.mean_lin, w.var_lin, ps, w.fused_ws, w.fused_bytes, st);
    if (rc) return rc;
    if (host_data_out && p1 > p0) {
      if (piped) {
        RSC_CUDA(cudaEventCreateWithFlags(&ev_cmp[c], cudaEventDisableTiming));
        RSC_CUDA(cudaEventRecord(ev_cmp[c], st));
        RSC_CUDA(cudaStreamWaitEvent(s_out, ev_cmp[c], 0));
      }
      RSC_CUDA(cudaMemcpyAsync(host_data_out + p0, h.data + p0, sizeof(float) * (size_t)(p1 - p0), cudaMemcpyDeviceToHost, s_out));
    }
  }
  host_chunk_reduce_kernel<<<(G + 255) / 256, 256, 0, st>>>(G, C, h.part_n_cells, h.part_total, h.part_sums,
                                                           h.o.gene_n_cells, h.o.gene_total_i64, h.sums);
  RSC_LAUNCH_CHECK("host_chunk_reduce_kernel");
  const size_t sG = (size_t)G;
  if (prm->which_moments & RSC_MOMENTS_LOG)
    if ((rc = finalize_moments(G, n, prm->ddof, h.sums, h.sums + sG, h.o.mean_log, h.o.var_log, st))) return rc;
  if (prm->which_moments & RSC_MOMENTS_LIN)
    if ((rc = finalize_moments(G, n, prm->ddof, h.sums + 2 * sG, h.sums + 3 * sG, h.o.mean_lin, h.o.var_lin, st))) return rc;
  {
    const double* hm = prm->hvg_on_linear ? h.o.mean_lin : h.o.mean_log;
    const double* hv = prm->hvg_on_linear ? h.o.var_lin : h.o.var_log;
    rc = launch_hvg(G, hm, hv, prm->n_top, prm->n_bins, prm->hvg_flags, h.o.hvg_mean_t, h.o.hvg_disp,
                    h.o.hvg_disp_norm, h.o.hvg_bin, h.o.hvg_mask, h.o.hvg_indices, h.o.hvg_count, w.hvg_ws,
                    w.hvg_bytes, st);
    if (rc) return rc;
  }
  if (piped) {                                             // join: the caller's stream also waits for the copies out
    RSC_CUDA(cudaEventRecord(ev_out, s_out));
    RSC_CUDA(cudaStreamWaitEvent(st, ev_out, 0));
    for (int c = 0; c < C; ++c) {
      if (ev_in[c]) cudaEventDestroy(ev_in[c]);            // released by the runtime once they have completed
      if (ev_cmp[c]) cudaEventDestroy(ev_cmp[c]);
    }
    cudaEventDestroy(ev_fork);
    cudaEventDestroy(ev_out);
  }
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
  return RSC_OK;
}

}  // extern "C"
