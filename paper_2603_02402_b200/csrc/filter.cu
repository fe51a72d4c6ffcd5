// filter_cells / filter_genes / HVG column subsetting.
//   rsc_filter_masks   keep-masks from the QC outputs and thresholds ("filtering",
//                      PAPER.md:L17, L21; thresholds = scanpy's filter_cells / filter_genes)
//   rsc_subset_csr_*   X[keep_rows][:, keep_cols] as a new CSR with a rebuilt int64 indptr:
//                      plan (column map, kept entries per row, device-wide scan -> out_indptr
//                      and the three output sizes) then fill (ordered compaction, warp per row).
// Same streaming regime as the rest of the path: plan reads indices (4 B / nnz), fill reads
// indices + data (8 B / nnz) and writes 8 B per kept entry.
#include <math.h>

#include "common.cuh"

namespace rsc {

constexpr int kScanBlock = 1024;            // rows per block of the device-wide scan

// ------------------------------------------------------------------ masks
__global__ void __launch_bounds__(256)
filter_masks_kernel(int64_t n_rows, int32_t n_cols, const int32_t* __restrict__ cell_n_genes,
                    const int64_t* __restrict__ cell_total, const float* __restrict__ cell_pct,
                    const int32_t* __restrict__ gene_n_cells, const int64_t* __restrict__ gene_total,
                    rsc_filter_params p, uint8_t* __restrict__ cell_keep, uint8_t* __restrict__ gene_keep) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t nth = (int64_t)gridDim.x * blockDim.x;
  if (cell_keep != nullptr) {
    for (int64_t i = t; i < n_rows; i += nth) {
      bool k = true;
      if (cell_n_genes) k = k && cell_n_genes[i] >= p.min_genes;
      if (cell_total) k = k && cell_total[i] >= p.min_counts;
      if (cell_pct && isfinite(p.max_pct_flag)) k = k && (cell_pct[i] <= p.max_pct_flag);   // NaN fails
      cell_keep[i] = k ? 1 : 0;
    }
  }
  if (gene_keep != nullptr) {
    for (int64_t j = t; j < n_cols; j += nth) {
      bool k = true;
      if (gene_n_cells) k = k && gene_n_cells[j] >= p.min_cells;
      if (gene_total) k = k && gene_total[j] >= p.min_gene_counts;
      gene_keep[j] = k ? 1 : 0;
    }
  }
}

int launch_filter_masks(int64_t n_rows, int32_t n_cols, const int32_t* cell_n_genes,
                        const int64_t* cell_total, const float* cell_pct, const int32_t* gene_n_cells,
                        const int64_t* gene_total, const rsc_filter_params& p, uint8_t* cell_keep,
                        uint8_t* gene_keep, cudaStream_t st) {
  int64_t work = n_rows > n_cols ? n_rows : n_cols;
  if (work <= 0) return RSC_OK;
  int64_t blocks = (work + 255) / 256;
  const int64_t cap = (int64_t)sm_count() * 8;
  if (blocks > cap) blocks = cap;
  filter_masks_kernel<<<(unsigned)blocks, 256, 0, st>>>(n_rows, n_cols, cell_n_genes, cell_total, cell_pct,
                                                        gene_n_cells, gene_total, p, cell_keep, gene_keep);
  RSC_LAUNCH_CHECK("filter_masks_kernel");
  return RSC_OK;
}

// ------------------------------------------------------------------ subset: workspace
struct SubsetWs {
  int32_t* col_map;          // [n_cols] new column index or -1
  int64_t* row_off;          // [n_rows] offset of the row in the output (kept rows)
  uint32_t* row_cnt;         // [n_rows] kept entries of the row (0 for dropped rows)
  int64_t* blk;              // [2 * n_blocks] per scan block: kept rows, kept entries (then exclusive)
  int64_t* meta;             // [3] copy of out_counts (kept rows, kept columns, kept entries) for the fill call
  size_t total;
};

static SubsetWs carve_subset(void* ws, int64_t n_rows, int32_t n_cols) {
  unsigned char* b = static_cast<unsigned char*>(ws);
  SubsetWs w;
  size_t o = 0;
  const size_t nb = (size_t)((n_rows + kScanBlock - 1) / kScanBlock);
  w.col_map = reinterpret_cast<int32_t*>(b + o);  o += align_up(sizeof(int32_t) * (size_t)n_cols, 256);
  w.row_off = reinterpret_cast<int64_t*>(b + o);  o += align_up(sizeof(int64_t) * (size_t)n_rows, 256);
  w.row_cnt = reinterpret_cast<uint32_t*>(b + o); o += align_up(sizeof(uint32_t) * (size_t)n_rows, 256);
  w.blk = reinterpret_cast<int64_t*>(b + o);      o += align_up(sizeof(int64_t) * 2 * (nb + 1), 256);
  w.meta = reinterpret_cast<int64_t*>(b + o);     o += 256;
  w.total = o;
  return w;
}

size_t subset_workspace_bytes(int64_t n_rows, int32_t n_cols) {
  return carve_subset(nullptr, n_rows < 0 ? 0 : n_rows, n_cols < 0 ? 0 : n_cols).total;
}

// ------------------------------------------------------------------ subset: plan kernels
// column map by one CTA: chunks of 1024 columns, ballot + warp counts, running base
__global__ void __launch_bounds__(1024)
subset_colmap_kernel(int32_t n_cols, const uint8_t* __restrict__ keep_cols, int32_t* __restrict__ col_map,
                     int64_t* __restrict__ out_counts, int64_t* __restrict__ meta) {
  __shared__ int wsum[32];
  __shared__ int s_base;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) s_base = 0;
  __syncthreads();
  for (int c0 = 0; c0 < n_cols; c0 += 1024) {
    const int c = c0 + tid;
    const bool k = c < n_cols && (keep_cols == nullptr || keep_cols[c] != 0);
    const unsigned bal = __ballot_sync(0xffffffffu, k);
    if (lane == 0) wsum[warp] = __popc(bal);
    __syncthreads();
    int off = s_base;
    for (int w = 0; w < warp; ++w) off += wsum[w];
    if (c < n_cols) col_map[c] = k ? off + __popc(bal & ((1u << lane) - 1u)) : -1;
    __syncthreads();
    if (tid == 0) { int t = s_base; for (int w = 0; w < 32; ++w) t += wsum[w]; s_base = t; }
    __syncthreads();
  }
  if (tid == 0) { out_counts[1] = s_base; meta[1] = s_base; }
}

// kept entries per row (warp per row; dropped rows count 0).  When every column is kept (the
// column map's kept count, already on the device, equals n_cols: a pure row filter) the count is
// the row length and the indices are not read at all.  (128-bit quad loads were measured slower
// than four independent 4-byte loads per lane here: the column-map gathers dominate.)
__global__ void __launch_bounds__(256)
subset_count_kernel(int64_t n_rows, int64_t nnz, int32_t n_cols, const int64_t* __restrict__ indptr,
                    const int32_t* __restrict__ indices, const uint8_t* __restrict__ keep_rows,
                    const int32_t* __restrict__ col_map, const int64_t* __restrict__ out_counts,
                    uint32_t* __restrict__ row_cnt) {
  const int lane = lane_id();
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const bool all_cols = out_counts[1] == (int64_t)n_cols;
  if (all_cols) {
    for (int64_t row = warp0 * 32 + lane; row < n_rows; row += nwarps * 32) {
      const bool k = keep_rows == nullptr || keep_rows[row] != 0;
      row_cnt[row] = k ? (uint32_t)(indptr[row + 1] - indptr[row]) : 0u;
    }
    return;
  }
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    unsigned c = 0;
    if (keep_rows == nullptr || keep_rows[row] != 0) {
      const int64_t beg = indptr[row], end = indptr[row + 1];
      for (int64_t p0 = beg; p0 < end; p0 += 128) {       // 4 independent loads per lane in flight
        int j[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const int64_t p = p0 + u * 32 + lane; j[u] = p < end ? __ldg(indices + p) : -1; }
#pragma unroll
        for (int u = 0; u < 4; ++u) c += (j[u] >= 0 && col_map[j[u]] >= 0) ? 1u : 0u;
      }
    }
    c = warp_sum(c);
    if (lane == 0) row_cnt[row] = c;
  }
}

// per scan block: number of kept rows and kept entries
__global__ void __launch_bounds__(kScanBlock)
subset_blocksum_kernel(int64_t n_rows, const uint8_t* __restrict__ keep_rows,
                       const uint32_t* __restrict__ row_cnt, int64_t* __restrict__ blk) {
  __shared__ long long s_r[32], s_e[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t row = (int64_t)blockIdx.x * kScanBlock + tid;
  long long r = 0, e = 0;
  if (row < n_rows && (keep_rows == nullptr || keep_rows[row] != 0)) { r = 1; e = row_cnt[row]; }
  r = warp_sum(r); e = warp_sum(e);
  if (lane == 0) { s_r[warp] = r; s_e[warp] = e; }
  __syncthreads();
  if (tid == 0) {
    long long tr = 0, te = 0;
    for (int w = 0; w < 32; ++w) { tr += s_r[w]; te += s_e[w]; }
    blk[2 * blockIdx.x] = tr; blk[2 * blockIdx.x + 1] = te;
  }
}

// exclusive scan of the block sums by one CTA; totals -> out_counts[0] (rows), [2] (entries)
__global__ void __launch_bounds__(1024)
subset_blockscan_kernel(int64_t n_blocks, int64_t* __restrict__ blk, int64_t* __restrict__ out_counts) {
  __shared__ long long s_r[32], s_e[32];
  __shared__ long long base_r, base_e;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) { base_r = 0; base_e = 0; }
  __syncthreads();
  for (int64_t b0 = 0; b0 < n_blocks; b0 += 1024) {
    const int64_t b = b0 + tid;
    long long r = b < n_blocks ? blk[2 * b] : 0, e = b < n_blocks ? blk[2 * b + 1] : 0;
    long long ir = r, ie = e;                              // inclusive warp scan
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const long long tr = __shfl_up_sync(0xffffffffu, ir, o), te = __shfl_up_sync(0xffffffffu, ie, o);
      if (lane >= o) { ir += tr; ie += te; }
    }
    if (lane == 31) { s_r[warp] = ir; s_e[warp] = ie; }
    __syncthreads();
    long long or_ = base_r, oe = base_e;
    for (int w = 0; w < warp; ++w) { or_ += s_r[w]; oe += s_e[w]; }
    if (b < n_blocks) { blk[2 * b] = or_ + ir - r; blk[2 * b + 1] = oe + ie - e; }
    __syncthreads();
    if (tid == 0) { for (int w = 0; w < 32; ++w) { base_r += s_r[w]; base_e += s_e[w]; } }
    __syncthreads();
  }
  if (tid == 0) { out_counts[0] = base_r; out_counts[2] = base_e; }
}

// block-local exclusive scan + block base: out_indptr[rank] = offset, row_off[row] = offset
__global__ void __launch_bounds__(kScanBlock)
subset_offsets_kernel(int64_t n_rows, const uint8_t* __restrict__ keep_rows,
                      const uint32_t* __restrict__ row_cnt, const int64_t* __restrict__ blk,
                      const int64_t* __restrict__ out_counts, int64_t* __restrict__ row_off,
                      int64_t* __restrict__ out_indptr) {
  __shared__ long long s_r[32], s_e[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t row = (int64_t)blockIdx.x * kScanBlock + tid;
  const bool k = row < n_rows && (keep_rows == nullptr || keep_rows[row] != 0);
  const long long r = k ? 1 : 0, e = k ? (long long)row_cnt[row] : 0;
  long long ir = r, ie = e;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const long long tr = __shfl_up_sync(0xffffffffu, ir, o), te = __shfl_up_sync(0xffffffffu, ie, o);
    if (lane >= o) { ir += tr; ie += te; }
  }
  if (lane == 31) { s_r[warp] = ir; s_e[warp] = ie; }
  __syncthreads();
  long long or_ = blk[2 * blockIdx.x], oe = blk[2 * blockIdx.x + 1];
  for (int w = 0; w < warp; ++w) { or_ += s_r[w]; oe += s_e[w]; }
  if (k) {
    const long long rank = or_ + ir - r, off = oe + ie - e;
    row_off[row] = off;
    out_indptr[rank] = off;
  }
  if (row == n_rows - 1 || (n_rows == 0 && blockIdx.x == 0 && tid == 0)) out_indptr[out_counts[0]] = out_counts[2];
}

// ------------------------------------------------------------------ subset: fill (warp per kept row)
// Every column kept (pure row filter): the kept rows are copied as they are.  Otherwise an
// ordered warp compaction (ballot prefix) through the column map.
__global__ void __launch_bounds__(256)
subset_fill_kernel(int64_t n_rows, int32_t n_cols, const int64_t* __restrict__ indptr,
                   const int32_t* __restrict__ indices, const float* __restrict__ data,
                   const uint8_t* __restrict__ keep_rows, const int32_t* __restrict__ col_map,
                   const int64_t* __restrict__ row_off, const int64_t* __restrict__ out_counts,
                   int32_t* __restrict__ out_indices, float* __restrict__ out_data) {
  const int lane = lane_id();
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const bool all_cols = out_counts[1] == (int64_t)n_cols;
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    if (keep_rows != nullptr && keep_rows[row] == 0) continue;
    const int64_t beg = indptr[row], end = indptr[row + 1];
    int64_t o = row_off[row];
    if (all_cols) {
      for (int64_t p0 = beg; p0 < end; p0 += 256) {       // 8 independent loads per lane and array in flight
        int j[8];
        float x[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const int64_t p = p0 + u * 32 + lane;
          j[u] = p < end ? __ldg(indices + p) : 0;
          x[u] = p < end ? __ldg(data + p) : 0.0f;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const int64_t p = p0 + u * 32 + lane;
          if (p < end) { out_indices[o + (p - beg)] = j[u]; out_data[o + (p - beg)] = x[u]; }
        }
      }
      continue;
    }
    for (int64_t p0 = beg; p0 < end; p0 += 128) {         // 4 independent loads per lane in flight
      int j[4];
      float x[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int64_t p = p0 + u * 32 + lane;
        j[u] = p < end ? __ldg(indices + p) : -1;
        x[u] = p < end ? __ldg(data + p) : 0.0f;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int jn = j[u] >= 0 ? col_map[j[u]] : -1;
        const unsigned bal = __ballot_sync(0xffffffffu, jn >= 0);
        if (jn >= 0) {
          const int64_t q = o + __popc(bal & ((1u << lane) - 1u));
          out_indices[q] = jn;
          out_data[q] = x[u];
        }
        o += __popc(bal);
      }
    }
  }
}

// ------------------------------------------------------------------ launchers
int launch_subset_plan(const rsc_csr& X, const uint8_t* keep_rows, const uint8_t* keep_cols,
                       int64_t* out_indptr, int64_t* out_counts, void* ws, cudaStream_t st) {
  SubsetWs w = carve_subset(ws, X.n_rows, X.n_cols);
  subset_colmap_kernel<<<1, 1024, 0, st>>>(X.n_cols, keep_cols, w.col_map, out_counts, w.meta);
  RSC_LAUNCH_CHECK("subset_colmap_kernel");
  const int64_t n = X.n_rows;
  const int64_t nb = (n + kScanBlock - 1) / kScanBlock;
  if (n > 0) {
    int64_t blocks = (n + 7) / 8;
    const int64_t cap = (int64_t)sm_count() * 16;
    if (blocks > cap) blocks = cap;
    subset_count_kernel<<<(unsigned)blocks, 256, 0, st>>>(n, X.nnz, X.n_cols, X.indptr, X.indices, keep_rows, w.col_map,
                                                          w.meta, w.row_cnt);
    RSC_LAUNCH_CHECK("subset_count_kernel");
    subset_blocksum_kernel<<<(unsigned)nb, kScanBlock, 0, st>>>(n, keep_rows, w.row_cnt, w.blk);
    RSC_LAUNCH_CHECK("subset_blocksum_kernel");
  }
  subset_blockscan_kernel<<<1, 1024, 0, st>>>(nb, w.blk, out_counts);
  RSC_LAUNCH_CHECK("subset_blockscan_kernel");
  subset_offsets_kernel<<<(unsigned)(nb > 0 ? nb : 1), kScanBlock, 0, st>>>(n, keep_rows, w.row_cnt, w.blk,
                                                                         out_counts, w.row_off, out_indptr);
  RSC_LAUNCH_CHECK("subset_offsets_kernel");
  return RSC_OK;
}

int launch_subset_fill(const rsc_csr& X, const uint8_t* keep_rows, int32_t* out_indices, float* out_data,
                       void* ws, cudaStream_t st) {
  if (X.n_rows == 0 || X.nnz == 0) return RSC_OK;
  SubsetWs w = carve_subset(ws, X.n_rows, X.n_cols);
  int64_t blocks = (X.n_rows + 7) / 8;
  const int64_t cap = (int64_t)sm_count() * 16;
  if (blocks > cap) blocks = cap;
  subset_fill_kernel<<<(unsigned)blocks, 256, 0, st>>>(X.n_rows, X.n_cols, X.indptr, X.indices, X.data, keep_rows,
                                                       w.col_map, w.row_off, w.meta, out_indices, out_data);
  RSC_LAUNCH_CHECK("subset_fill_kernel");
  return RSC_OK;
}

}  // namespace rsc

// ------------------------------------------------------------------ NEXT-4 (part): HVG by cutoffs
// mask_j = min_mean < m_j < max_mean and min_disp < z_j < max_disp (strict; NaN fails), the
// selected genes listed in ascending order (one CTA: chunks of 1024 genes, ballot + running base)
namespace rsc {

__global__ void __launch_bounds__(1024)
hvg_cutoffs_kernel(int32_t G, const double* __restrict__ mean_t, const double* __restrict__ disp_norm,
                   double min_mean, double max_mean, double min_disp, double max_disp,
                   uint8_t* __restrict__ out_mask, int32_t* __restrict__ out_idx, int32_t* __restrict__ out_count) {
  __shared__ int wsum[32];
  __shared__ int s_base;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) s_base = 0;
  __syncthreads();
  for (int c0 = 0; c0 < G; c0 += 1024) {
    const int g = c0 + tid;
    bool k = false;
    if (g < G) {
      const double m = mean_t[g], z = disp_norm[g];
      k = m > min_mean && m < max_mean && z > min_disp && z < max_disp;
      out_mask[g] = k ? 1 : 0;
    }
    const unsigned bal = __ballot_sync(0xffffffffu, k);
    if (lane == 0) wsum[warp] = __popc(bal);
    __syncthreads();
    int off = s_base;
    for (int w = 0; w < warp; ++w) off += wsum[w];
    if (k && out_idx != nullptr) out_idx[off + __popc(bal & ((1u << lane) - 1u))] = g;
    __syncthreads();
    if (tid == 0) { int t = s_base; for (int w = 0; w < 32; ++w) t += wsum[w]; s_base = t; }
    __syncthreads();
  }
  if (tid == 0) *out_count = s_base;
}

int launch_hvg_cutoffs(int32_t G, const double* mean_t, const double* disp_norm, double min_mean,
                       double max_mean, double min_disp, double max_disp, uint8_t* out_mask,
                       int32_t* out_idx, int32_t* out_count, cudaStream_t st) {
  hvg_cutoffs_kernel<<<1, 1024, 0, st>>>(G, mean_t, disp_norm, min_mean, max_mean, min_disp, max_disp,
                                         out_mask, out_idx, out_count);
  RSC_LAUNCH_CHECK("hvg_cutoffs_kernel");
  return RSC_OK;
}

}  // namespace rsc
