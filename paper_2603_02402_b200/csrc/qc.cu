// rsc_qc_metrics, streaming kernel ("QC metrics", cell-wise on CSR; L17/L21
// "filtering").  One pass over indices + data (8 B / nnz):
//   * per-cell sums by a warp per row (dynamic row grabs, so skewed row lengths balance);
//   * per-gene counts / totals in a CTA-private shared-memory table updated with native
//     32-bit shared atomics (ATOMS.ADD): total_j as a u32 word whose carries go straight to
//     the 64-bit global output, n_cells_j as a 16-bit field (two genes per word).  A CTA
//     flushes its table after at most row_budget + 4 (< 2^16) rows, so a field cannot wrap;
//   * optionally the row split table consumed by the fused pass (fused.cu): for every row,
//     the number of entries with column < k * RSC_SPLIT_WIDTH, found by comparing the
//     column block of neighbouring entries (rows must be sorted for the table to be valid).
// Genes that do not fit the shared-memory table (n_cols > ~37 k) fall back to L2 atomics.
#include "common.cuh"

namespace rsc {

constexpr int kQcThreads = 1024;
constexpr int kQcWarps = kQcThreads / 32;
constexpr int kQcRowsPerGrab = 4;
constexpr int kQcUnroll = 4;

struct QcArgs {
  int64_t n_rows;
  int32_t n_cols;
  int32_t n_smem_genes;      // genes [0, n_smem_genes) accumulate in shared memory
  int32_t n_fine;            // K = number of column blocks (split table has K + 1 entries per row)
  int32_t want_gene;         // gene_n_cells or gene_total requested
  uint32_t row_budget;       // a CTA stops grabbing rows once it has taken this many (then flushes)
  const int64_t* indptr;
  const int32_t* indices;
  const float* data;
  const uint8_t* flags;
  int64_t* cell_total;
  float* cell_total_f32;
  int32_t* cell_n_genes;
  int64_t* cell_flag_total;
  float* cell_flag_pct;
  int32_t* gene_n_cells;
  unsigned long long* gene_total;
  uint32_t* splits;
  unsigned long long* row_counter;
};

__device__ __forceinline__ long long warp_sum_ll(long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(kQcThreads, 1) qc_stream_kernel(const QcArgs a) {
  extern __shared__ __align__(16) uint32_t qsm[];
  const int Gs = a.n_smem_genes;
  uint32_t* tot = qsm;                                  // [Gs]
  uint32_t* cnt = tot + Gs;                             // [(Gs + 1) / 2], 16-bit fields
  uint32_t* fbits = cnt + ((Gs + 1) >> 1);              // [(G + 31) / 32]
  const int nfw = (a.n_cols + 31) >> 5;
  const int tid = threadIdx.x, lane = tid & 31;
  const bool has_flags = a.flags != nullptr;
  const bool want_gene = a.want_gene != 0;

  __shared__ unsigned s_rows;
  for (int i = tid; i < Gs + ((Gs + 1) >> 1); i += kQcThreads) qsm[i] = 0u;
  if (has_flags) {
    for (int g0 = (tid >> 5) << 5; g0 < a.n_cols; g0 += kQcThreads) {
      const int g = g0 + lane;
      const unsigned b = __ballot_sync(0xffffffffu, g < a.n_cols && a.flags[g] != 0);
      if (lane == 0) fbits[g0 >> 5] = b;
    }
  } else {
    for (int i = tid; i < nfw; i += kQcThreads) fbits[i] = 0u;
  }

  const int K = a.n_fine;
  const bool want_splits = a.splits != nullptr;

  // -1: the CTA's row budget is used up (flush first); >= n_rows: the matrix is exhausted
  // (only lane 0 holds the result; it is broadcast when needed, so the L2 round trip of the
  // atomic overlaps the rows being processed)
  auto grab_issue = [&]() -> long long {
    long long r = -1;
    if (lane == 0) {
      const unsigned c = atomicAdd(&s_rows, (unsigned)kQcRowsPerGrab);
      if (c < a.row_budget)
        r = (long long)atomicAdd(a.row_counter, (unsigned long long)kQcRowsPerGrab);
    }
    return r;
  };

  int done;
  do {
    if (tid == 0) s_rows = 0u;
    __syncthreads();
    int saw_end = 0;
    long long r0 = __shfl_sync(0xffffffffu, grab_issue(), 0);
    while (r0 >= 0) {
      if (r0 >= a.n_rows) { saw_end = 1; break; }
      const long long pending = grab_issue();
      const long long rend = min((long long)a.n_rows, r0 + kQcRowsPerGrab);
      for (long long row = r0; row < rend; ++row) {
        const int64_t beg = a.indptr[row], end = a.indptr[row + 1];
        long long T = 0, M = 0;
        int N = 0;
        int carry_f = -1;                                // column block of the previous entry
        uint32_t* sp = want_splits ? a.splits + (size_t)row * (size_t)(K + 1) : nullptr;
        for (int64_t base = beg; base < end; base += 32 * kQcUnroll) {
          int j[kQcUnroll];
          float x[kQcUnroll];
#pragma unroll
          for (int u = 0; u < kQcUnroll; ++u) {
            const int64_t p = base + u * 32 + lane;
            const bool ok = p < end;
            j[u] = ok ? __ldg(a.indices + p) : -1;
            x[u] = ok ? __ldg(a.data + p) : 0.0f;
          }
#pragma unroll
          for (int u = 0; u < kQcUnroll; ++u) {
            const int jj = j[u];
            const bool ok = jj >= 0;
            if (want_splits) {
              const int f = ok ? (jj >> RSC_SPLIT_SHIFT) : K;
              int fp = __shfl_up_sync(0xffffffffu, f, 1);
              if (lane == 0) fp = carry_f;
              carry_f = __shfl_sync(0xffffffffu, f, 31);
              if (f > fp) {
                const int64_t p = base + u * 32 + lane;
                const uint32_t pos = (uint32_t)((p < end ? p : end) - beg);
                for (int k = fp + 1; k <= f; ++k) sp[k] = pos;
              }
            }
            if (ok) {
              const float xv = x[u];
              const long long xi = (long long)xv;
              const bool nz = xv != 0.0f;
              T += xi;
              N += nz;
              if (has_flags && ((fbits[jj >> 5] >> (jj & 31)) & 1u)) M += xi;
              if (want_gene) {
                if (jj < Gs && xi >= 0 && xi <= 0x7fffffffLL) {
                  const uint32_t xu = (uint32_t)xi;
                  if (xu != 0u) {
                    const uint32_t old = atomicAdd(&tot[jj], xu);
                    if (old + xu < old && a.gene_total != nullptr)   // carry out of the u32 word
                      atomicAdd(&a.gene_total[jj], 1ull << 32);
                  }
                  if (nz) atomicAdd(&cnt[jj >> 1], 1u << ((jj & 1) << 4));
                } else {
                  if (nz && a.gene_n_cells != nullptr) atomicAdd(&a.gene_n_cells[jj], 1);
                  if (xi != 0 && a.gene_total != nullptr)
                    atomicAdd(&a.gene_total[jj], (unsigned long long)xi);
                }
              }
            }
          }
        }
        if (want_splits) {
          const uint32_t len = (uint32_t)(end - beg);
          for (int k = carry_f + 1 + lane; k <= K; k += 32) sp[k] = len;
        }
        T = warp_sum_ll(T);
        M = warp_sum_ll(M);
        N = warp_sum(N);
        if (lane == 0) {
          if (a.cell_total) a.cell_total[row] = T;
          if (a.cell_total_f32) a.cell_total_f32[row] = (float)T;
          if (a.cell_n_genes) a.cell_n_genes[row] = N;
          if (a.cell_flag_total) a.cell_flag_total[row] = M;
          if (a.cell_flag_pct) a.cell_flag_pct[row] = (float)(100.0 * (double)M / (double)T);
        }
      }
      r0 = __shfl_sync(0xffffffffu, pending, 0);
    }
    done = __syncthreads_or(saw_end);
    if (want_gene) {                                     // flush and clear the CTA's table
      for (int g = tid; g < Gs; g += kQcThreads) {
        const uint32_t t = tot[g];
        if (t != 0u) {
          if (a.gene_total != nullptr) atomicAdd(&a.gene_total[g], (unsigned long long)t);
          tot[g] = 0u;
        }
      }
      for (int w = tid; w < ((Gs + 1) >> 1); w += kQcThreads) {
        const uint32_t c = cnt[w];
        if (c != 0u) {
          if (a.gene_n_cells != nullptr) {
            if (c & 0xffffu) atomicAdd(&a.gene_n_cells[2 * w], (int)(c & 0xffffu));
            if (c >> 16) atomicAdd(&a.gene_n_cells[2 * w + 1], (int)(c >> 16));
          }
          cnt[w] = 0u;
        }
      }
    }
  } while (!done);
}

// ------------------------------------------------------------------ standalone split table
// splits[row * (K + 1) + k] = #{entries of the row with column < k * RSC_SPLIT_WIDTH}; one
// thread per (row, k), binary search in the (sorted) row.
__global__ void __launch_bounds__(256)
row_splits_kernel(int64_t n_rows, int K, const int64_t* __restrict__ indptr,
                  const int32_t* __restrict__ indices, uint32_t* __restrict__ splits) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t total = n_rows * (int64_t)(K + 1);
  if (t >= total) return;
  const int64_t row = t / (K + 1);
  const int k = (int)(t - row * (K + 1));
  const int64_t beg = indptr[row], end = indptr[row + 1];
  const int32_t bound = k << RSC_SPLIT_SHIFT;
  int64_t lo = beg, hi = end;
  if (k == 0) hi = beg;
  else if (k == K) lo = end;
  while (lo < hi) {
    const int64_t mid = (lo + hi) >> 1;
    if (__ldg(indices + mid) < bound) lo = mid + 1; else hi = mid;
  }
  splits[t] = (uint32_t)(lo - beg);
}

int launch_row_splits(const rsc_csr& X, uint32_t* splits, cudaStream_t st) {
  if (X.n_rows == 0) return RSC_OK;
  const int K = split_blocks(X.n_cols);
  const int64_t total = X.n_rows * (int64_t)(K + 1);
  const int64_t blocks = (total + 255) / 256;
  if (blocks > 0x7fffffffLL) {
    set_error("rsc_row_splits: matrix too large for the split kernel grid");
    return RSC_ERR_INVALID_ARG;
  }
  row_splits_kernel<<<(unsigned)blocks, 256, 0, st>>>(X.n_rows, K, X.indptr, X.indices, splits);
  RSC_LAUNCH_CHECK("row_splits_kernel");
  return RSC_OK;
}

// ------------------------------------------------------------------ launcher
size_t qc_workspace_bytes(int64_t, int32_t, int64_t) { return 256; }

static int qc_smem_genes(int32_t n_cols, size_t* smem_bytes) {
  const size_t fixed = sizeof(uint32_t) * (size_t)((n_cols + 31) / 32) + 64;
  size_t avail = kMaxDynSmem > fixed ? kMaxDynSmem - fixed : 0;
  // 4 bytes (total) + 2 bytes (count field) per gene
  long long gs = (long long)(avail / 6);
  gs &= ~1LL;
  if (gs > n_cols) gs = n_cols;
  if (gs < 0) gs = 0;
  *smem_bytes = sizeof(uint32_t) * ((size_t)gs + (size_t)((gs + 1) / 2)) + fixed;
  return (int)gs;
}

int launch_qc(const rsc_csr& X, const uint8_t* gene_flags, int64_t* cell_total_i64,
              float* cell_total_f32, int32_t* cell_n_genes, int64_t* cell_flag_total_i64,
              float* cell_flag_pct, int32_t* gene_n_cells, int64_t* gene_total_i64,
              uint32_t* row_splits, void* ws, size_t, cudaStream_t st) {
  if (gene_n_cells) RSC_CUDA(cudaMemsetAsync(gene_n_cells, 0, sizeof(int32_t) * X.n_cols, st));
  if (gene_total_i64) RSC_CUDA(cudaMemsetAsync(gene_total_i64, 0, sizeof(int64_t) * X.n_cols, st));
  if (X.n_rows == 0) return RSC_OK;
  RSC_CUDA(cudaMemsetAsync(ws, 0, 256, st));
  QcArgs a;
  a.n_rows = X.n_rows;
  a.n_cols = X.n_cols;
  size_t smem = 0;
  a.n_smem_genes = qc_smem_genes(X.n_cols, &smem);
  a.n_fine = split_blocks(X.n_cols);
  a.want_gene = (gene_n_cells != nullptr || gene_total_i64 != nullptr) ? 1 : 0;
  a.indptr = X.indptr; a.indices = X.indices; a.data = X.data; a.flags = gene_flags;
  a.cell_total = cell_total_i64; a.cell_total_f32 = cell_total_f32; a.cell_n_genes = cell_n_genes;
  a.cell_flag_total = cell_flag_total_i64; a.cell_flag_pct = cell_flag_pct;
  a.gene_n_cells = gene_n_cells;
  a.gene_total = reinterpret_cast<unsigned long long*>(gene_total_i64);
  a.splits = row_splits;
  a.row_counter = static_cast<unsigned long long*>(ws);
  static bool attr_set = false;
  if (!attr_set) {
    RSC_CUDA(cudaFuncSetAttribute(qc_stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)kMaxDynSmem));
    attr_set = true;
  }
  a.row_budget = (uint32_t)g_opt.qc_row_budget;
  int64_t blocks = (X.n_rows + kQcWarps * kQcRowsPerGrab - 1) / (kQcWarps * kQcRowsPerGrab);
  const int cap = g_opt.grid_ctas > 0 ? g_opt.grid_ctas : sm_count();
  if (blocks > cap) blocks = cap;
  qc_stream_kernel<<<(unsigned)blocks, kQcThreads, smem, st>>>(a);
  RSC_LAUNCH_CHECK("qc_stream_kernel");
  return RSC_OK;
}

}  // namespace rsc
