// rsc_qc_metrics, streaming kernel ("QC metrics", cell-wise on CSR; L17/L21
// "filtering").  One pass over indices + data (8 B / nnz):
//   * per-cell sums by a warp per row (dynamic row grabs, so skewed row lengths balance);
//     a lane reads 4 consecutive entries with one 128-bit load per array;
//   * per-gene count AND total in ONE 32-bit word of a CTA-private shared-memory table,
//     updated with one native shared atomic (ATOMS.ADD) per stored entry:
//         bit 31      the gene's QC flag (set once; returned by the atomic, so the flagged
//                     subset total needs no second lookup)
//         bits 20..30 n_cells_j of this flush period   (11 bits)
//         bits 0..19  total_j of this flush period     (20 bits)
//     Entries with a count > 511 (or negative / beyond the table) bypass the table and go to
//     the global outputs directly.  A CTA flushes its table after at most 2047 rows
//     (2047 * 511 < 2^20), so no field can overflow into its neighbour;
//   * optionally the row split table consumed by the fused pass (fused.cu): for every row,
//     the number of entries with column < k * RSC_SPLIT_WIDTH, found by comparing the column
//     block of a lane's last entry with its neighbour's (rows must be sorted).
#include "common.cuh"

namespace rsc {

constexpr int kQcThreads = 1024;
constexpr int kQcWarps = kQcThreads / 32;
constexpr int kQcRowsPerGrab = 4;
constexpr int kQcUnroll = 2;                 // 2 x 128 entries per warp iteration
constexpr uint32_t kQcMaxFast = 511u;        // largest count that takes the shared-memory path
constexpr int kQcMaxRowBudget = 2047 - kQcRowsPerGrab;   // rows per flush period incl. the last grab

struct QcArgs {
  int64_t n_rows;
  int64_t nnz;
  int32_t n_cols;
  int32_t n_fine;            // K = number of column blocks (split table has K + 1 entries per row)
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

// shared-memory atomic add on a 32-bit shared address, executed only when `on` is set
// (a predicated ATOMS instead of a branch); returns the previous word (0 when skipped)
__device__ __forceinline__ uint32_t atoms_add_if(uint32_t saddr, uint32_t v, bool on) {
  uint32_t old = 0u;
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %3, 0;\n\t@p atom.shared.add.u32 %0, [%1], %2;\n\t}"
      : "+r"(old)
      : "r"(saddr), "r"(v), "r"((uint32_t)on)
      : "memory");
  return old;
}

template <bool SPLITS>
__global__ void __launch_bounds__(kQcThreads, 1) qc_stream_kernel(const QcArgs a) {
  extern __shared__ __align__(16) uint32_t qsm[];      // [G] packed flag | count | total
  const int G = a.n_cols;
  const int tid = threadIdx.x, lane = tid & 31;
  const int K = a.n_fine;
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(qsm);
  __shared__ unsigned s_rows;

  for (int g = tid; g < G; g += kQcThreads)
    qsm[g] = (a.flags != nullptr && a.flags[g] != 0) ? 0x80000000u : 0u;

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
      // lanes 0..RG fetch the row bounds of this grab
      int64_t mptr = 0;
      if (lane <= kQcRowsPerGrab && r0 + lane <= a.n_rows) mptr = a.indptr[r0 + lane];
      const int nr = (int)min((long long)kQcRowsPerGrab, a.n_rows - r0);
#pragma unroll 1
      for (int ri = 0; ri < nr; ++ri) {
        const long long row = r0 + ri;
        const int64_t beg = __shfl_sync(0xffffffffu, mptr, ri);
        const int64_t end = __shfl_sync(0xffffffffu, mptr, ri + 1);
        // all positions below are 32-bit offsets from the 4-aligned start of the row
        const int64_t abeg = beg & ~3LL;
        const int head = (int)(beg - abeg);             // entries of the previous row in the first quad
        const int len = (int)(end - beg);
        const int span = head + len;
        const int64_t room = a.nnz - abeg;              // a quad at offset r is a vector load iff r + 4 <= vlim
        const int vlim = room > 0x7fffffffLL ? 0x7fffffff : (int)room;
        const int32_t* ip = a.indices + abeg + lane * 4;
        const float* dp = a.data + abeg + lane * 4;
        unsigned t32 = 0, m32 = 0, n32 = 0;             // fast-path partial sums of this lane
        long long T64 = 0, M64 = 0;                     // slow-path (large / negative counts)
        int carry_f = -1;                               // column block of the previous entry
        uint32_t* sp = SPLITS ? a.splits + (size_t)row * (size_t)(K + 1) : nullptr;
        for (int rb = 0; rb < span; rb += 128 * kQcUnroll, ip += 128 * kQcUnroll, dp += 128 * kQcUnroll) {
          int j[kQcUnroll][4];
          float x[kQcUnroll][4];
#pragma unroll
          for (int u = 0; u < kQcUnroll; ++u) {
            const int r = rb + u * 128 + lane * 4;
            if (r + 4 <= vlim && r < span) {
              const int4 jv = __ldg(reinterpret_cast<const int4*>(ip + u * 128));
              const float4 xv = __ldg(reinterpret_cast<const float4*>(dp + u * 128));
              j[u][0] = jv.x; j[u][1] = jv.y; j[u][2] = jv.z; j[u][3] = jv.w;
              x[u][0] = xv.x; x[u][1] = xv.y; x[u][2] = xv.z; x[u][3] = xv.w;
            } else {
#pragma unroll
              for (int k = 0; k < 4; ++k) {             // last quad of the matrix, or past the row
                const bool ok = r + k < span && r + k < vlim;
                j[u][k] = ok ? __ldg(ip + u * 128 + k) : 0;
                x[u][k] = ok ? __ldg(dp + u * 128 + k) : 0.0f;
              }
            }
          }
#pragma unroll
          for (int u = 0; u < kQcUnroll; ++u) {
            const int e0 = rb + u * 128 + lane * 4 - head;   // row-relative index of the quad's first entry
            if (SPLITS) {
              // column block of every entry: -1 before the row, K after it
              int f[4];
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const int e = e0 + k;
                f[k] = e < 0 ? -1 : (e < len ? (j[u][k] >> RSC_SPLIT_SHIFT) : K);
              }
              int fp = __shfl_up_sync(0xffffffffu, f[3], 1);
              if (lane == 0) fp = carry_f;
              carry_f = __shfl_sync(0xffffffffu, f[3], 31);
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                if (f[k] != fp) {                       // first entry of block f[k] (and of skipped ones)
                  const uint32_t pos = (uint32_t)min(e0 + k, len);
#pragma unroll 1
                  for (int kk = fp + 1; kk <= f[k]; ++kk) sp[kk] = pos;
                }
                fp = f[k];
              }
            }
            bool any_slow = false;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const bool valid = (unsigned)(e0 + k) < (unsigned)len;
              const float xv = x[u][k];
              const int xi = __float2int_rz(xv);
              const bool nz = valid && xv != 0.0f;
              const bool fast = valid && (unsigned)xi <= kQcMaxFast;
              any_slow |= valid && !fast;
              const unsigned xf = fast ? (unsigned)xi : 0u;
              const uint32_t old =
                  atoms_add_if(sbase + ((uint32_t)j[u][k] << 2), xf + (nz ? 0x100000u : 0u), fast);
              n32 += nz ? 1u : 0u;
              t32 += xf;
              m32 += xf & (uint32_t)((int)old >> 31);
            }
            if (any_slow) {                             // rare: counts > 511, negative or non-finite values
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const bool valid = (unsigned)(e0 + k) < (unsigned)len;
                const float xv = x[u][k];
                if (!valid || (unsigned)__float2int_rz(xv) <= kQcMaxFast) continue;
                const int jj = j[u][k];
                const long long xl = (long long)xv;
                T64 += xl;
                if (qsm[jj] >> 31) M64 += xl;
                if (a.gene_n_cells != nullptr) atomicAdd(&a.gene_n_cells[jj], 1);
                if (xl != 0 && a.gene_total != nullptr)
                  atomicAdd(&a.gene_total[jj], (unsigned long long)xl);
              }
            }
          }
        }
        if (SPLITS) {
          for (int k = carry_f + 1 + lane; k <= K; k += 32) sp[k] = (uint32_t)len;
        }
        long long T, M;
        if (__any_sync(0xffffffffu, (T64 | M64) != 0)) {
          T = warp_sum_ll(T64 + (long long)t32);
          M = warp_sum_ll(M64 + (long long)m32);
        } else {                                        // 511 * len < 2^32: the 32-bit sums are exact
          T = (long long)warp_sum(t32);
          M = (long long)warp_sum(m32);
        }
        const int N = (int)warp_sum(n32);
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
    // flush and clear the CTA's table (the flag bit stays)
    for (int g = tid; g < G; g += kQcThreads) {
      const uint32_t w = qsm[g];
      const uint32_t c = (w >> 20) & 0x7ffu, t = w & 0xfffffu;
      if (c | t) {
        if (c != 0u && a.gene_n_cells != nullptr) atomicAdd(&a.gene_n_cells[g], (int)c);
        if (t != 0u && a.gene_total != nullptr) atomicAdd(&a.gene_total[g], (unsigned long long)t);
        qsm[g] = w & 0x80000000u;
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

// one packed word per gene must fit the CTA's shared memory (57 840 genes)
constexpr int kQcMaxGenes = (int)((kMaxDynSmem - 64) / sizeof(uint32_t));

int launch_qc_generic(const rsc_csr&, const uint8_t*, int64_t*, float*, int32_t*, int64_t*, float*,
                      int32_t*, int64_t*, cudaStream_t);

int launch_qc(const rsc_csr& X, const uint8_t* gene_flags, int64_t* cell_total_i64,
              float* cell_total_f32, int32_t* cell_n_genes, int64_t* cell_flag_total_i64,
              float* cell_flag_pct, int32_t* gene_n_cells, int64_t* gene_total_i64,
              uint32_t* row_splits, void* ws, size_t, cudaStream_t st) {
  // the 128-bit loads need 16-byte aligned arrays; anything else takes the generic kernel
  const bool aligned = ((reinterpret_cast<uintptr_t>(X.indices) | reinterpret_cast<uintptr_t>(X.data)) & 15) == 0;
  if (!aligned || g_opt.force_generic || X.n_cols > kQcMaxGenes) {
    int rc = launch_qc_generic(X, gene_flags, cell_total_i64, cell_total_f32, cell_n_genes,
                               cell_flag_total_i64, cell_flag_pct, gene_n_cells, gene_total_i64, st);
    if (rc != RSC_OK) return rc;
    if (row_splits != nullptr) return launch_row_splits(X, row_splits, st);
    return RSC_OK;
  }
  if (gene_n_cells) RSC_CUDA(cudaMemsetAsync(gene_n_cells, 0, sizeof(int32_t) * X.n_cols, st));
  if (gene_total_i64) RSC_CUDA(cudaMemsetAsync(gene_total_i64, 0, sizeof(int64_t) * X.n_cols, st));
  if (X.n_rows == 0) return RSC_OK;
  RSC_CUDA(cudaMemsetAsync(ws, 0, 256, st));
  QcArgs a;
  a.n_rows = X.n_rows;
  a.nnz = X.nnz;
  a.n_cols = X.n_cols;
  const size_t smem = sizeof(uint32_t) * (size_t)X.n_cols + 16;
  a.n_fine = split_blocks(X.n_cols);
  a.indptr = X.indptr; a.indices = X.indices; a.data = X.data; a.flags = gene_flags;
  a.cell_total = cell_total_i64; a.cell_total_f32 = cell_total_f32; a.cell_n_genes = cell_n_genes;
  a.cell_flag_total = cell_flag_total_i64; a.cell_flag_pct = cell_flag_pct;
  a.gene_n_cells = gene_n_cells;
  a.gene_total = reinterpret_cast<unsigned long long*>(gene_total_i64);
  a.splits = row_splits;
  a.row_counter = static_cast<unsigned long long*>(ws);
  static bool attr_set = false;
  if (!attr_set) {
    RSC_CUDA(cudaFuncSetAttribute(qc_stream_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)kMaxDynSmem));
    RSC_CUDA(cudaFuncSetAttribute(qc_stream_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)kMaxDynSmem));
    attr_set = true;
  }
  a.row_budget = (uint32_t)min(g_opt.qc_row_budget, kQcMaxRowBudget);
  int64_t blocks = (X.n_rows + kQcWarps * kQcRowsPerGrab - 1) / (kQcWarps * kQcRowsPerGrab);
  const int cap = g_opt.grid_ctas > 0 ? g_opt.grid_ctas : sm_count();
  if (blocks > cap) blocks = cap;
  if (row_splits != nullptr)
    qc_stream_kernel<true><<<(unsigned)blocks, kQcThreads, smem, st>>>(a);
  else
    qc_stream_kernel<false><<<(unsigned)blocks, kQcThreads, smem, st>>>(a);
  RSC_LAUNCH_CHECK("qc_stream_kernel");
  return RSC_OK;
}

}  // namespace rsc
