// Generic (order-agnostic) kernels: correct for any canonical CSR, including rows whose
// column indices are NOT sorted.  Per-gene sums go straight to L2 atomics, so these
// kernels are the fallback when RSC_CSR_SORTED is not set, and they also serve the
// unfused elementwise steps (normalize_total, log1p) whose cost is pure streaming.
//
// PAPER.md:L85 (QC metrics, cell-wise on CSR), L91 (normalize_total, log1p, per-gene
// mean/variance kernel "that operates directly on sparse matrices"), L135 ("scatter-add
// kernels with atomic operations").
#include "common.cuh"

namespace rsc {

// ------------------------------------------------------------------ QC, warp per row
__global__ void __launch_bounds__(256)
qc_generic_kernel(int64_t n_rows, const int64_t* __restrict__ indptr,
                  const int32_t* __restrict__ indices, const float* __restrict__ data,
                  const uint8_t* __restrict__ flags, int64_t* __restrict__ cell_total,
                  float* __restrict__ cell_total_f32, int32_t* __restrict__ cell_n_genes,
                  int64_t* __restrict__ cell_flag_total, float* __restrict__ cell_flag_pct,
                  int32_t* __restrict__ gene_n_cells,
                  unsigned long long* __restrict__ gene_total) {
  const int lane = lane_id();
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    const int64_t beg = indptr[row], end = indptr[row + 1];
    long long T = 0, M = 0;
    int N = 0;
    for (int64_t p = beg + lane; p < end; p += 32) {
      const float x = data[p];
      const int j = indices[p];
      const long long xi = (long long)x;
      const int nz = x != 0.0f;
      T += xi;
      N += nz;
      if (flags != nullptr && flags[j]) M += xi;
      if (gene_n_cells != nullptr && nz) atomicAdd(&gene_n_cells[j], 1);
      if (gene_total != nullptr && xi != 0) atomicAdd(&gene_total[j], (unsigned long long)xi);
    }
    T = warp_sum(T);
    M = warp_sum(M);
    N = warp_sum(N);
    if (lane == 0) {
      if (cell_total) cell_total[row] = T;
      if (cell_total_f32) cell_total_f32[row] = (float)T;
      if (cell_n_genes) cell_n_genes[row] = N;
      if (cell_flag_total) cell_flag_total[row] = M;
      if (cell_flag_pct) cell_flag_pct[row] = (float)(100.0 * (double)M / (double)T);
    }
  }
}

int launch_qc_generic(const rsc_csr& X, const uint8_t* gene_flags, int64_t* cell_total_i64,
                      float* cell_total_f32, int32_t* cell_n_genes, int64_t* cell_flag_total_i64,
                      float* cell_flag_pct, int32_t* gene_n_cells, int64_t* gene_total_i64,
                      cudaStream_t st) {
  if (gene_n_cells) RSC_CUDA(cudaMemsetAsync(gene_n_cells, 0, sizeof(int32_t) * X.n_cols, st));
  if (gene_total_i64) RSC_CUDA(cudaMemsetAsync(gene_total_i64, 0, sizeof(int64_t) * X.n_cols, st));
  if (X.n_rows == 0) return RSC_OK;
  const int threads = 256;
  int64_t blocks = (X.n_rows + 7) / 8;
  const int64_t cap = (int64_t)sm_count() * 8;
  if (blocks > cap) blocks = cap;
  qc_generic_kernel<<<(unsigned)blocks, threads, 0, st>>>(
      X.n_rows, X.indptr, X.indices, X.data, gene_flags, cell_total_i64, cell_total_f32,
      cell_n_genes, cell_flag_total_i64, cell_flag_pct, gene_n_cells,
      reinterpret_cast<unsigned long long*>(gene_total_i64));
  RSC_LAUNCH_CHECK("qc_generic_kernel");
  return RSC_OK;
}

// ------------------------------------------------------------------ normalize_total
// x' = x * scale_i in place: 4 B read + 4 B written per stored entry.  A warp per
// row; the row is walked as 16-byte aligned float4's (scalar head / tail of at most 3
// elements), four per lane in flight.  Without supplied totals the row is summed first (fp64;
// the second sweep finds it in L1 / L2).
__device__ __forceinline__ void row_vec_bounds(const float* rowp, int64_t len, int& head, int64_t& nvec) {
  const uintptr_t a = reinterpret_cast<uintptr_t>(rowp);
  const int64_t h = ((16 - (a & 15)) & 15) >> 2;
  head = (int)(h < len ? h : len);
  nvec = (len - head) >> 2;
}

__global__ void __launch_bounds__(256)
normalize_kernel(int64_t n_rows, const int64_t* __restrict__ indptr, float* __restrict__ data,
                 float target_sum, const int64_t* __restrict__ cell_total,
                 float* __restrict__ scale_out) {
  const int lane = lane_id();
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    const int64_t beg = indptr[row], len = indptr[row + 1] - beg;
    float* rowp = data + beg;
    int head;
    int64_t nvec;
    row_vec_bounds(rowp, len, head, nvec);
    float4* vp = reinterpret_cast<float4*>(rowp + head);
    const int64_t tail0 = head + (nvec << 2);
    float scale;
    if (cell_total != nullptr) {
      scale = cell_scale(target_sum, cell_total[row]);
    } else {
      double s = 0.0;
      if (lane < head) s += (double)rowp[lane];
      for (int64_t i = lane; i < nvec; i += 32) {
        const float4 v = vp[i];
        s += ((double)v.x + (double)v.y) + ((double)v.z + (double)v.w);
      }
      if (tail0 + lane < len) s += (double)rowp[tail0 + lane];
      s = warp_sum(s);
      const float sf = (float)s;
      scale = sf != 0.0f ? __fdiv_rn(target_sum, sf) : 1.0f;
    }
    if (lane < head) rowp[lane] = __fmul_rn(rowp[lane], scale);
    int64_t i = lane;
    for (; i + 96 < nvec; i += 128) {                     // four loads in flight per lane
      float4 a = vp[i], b = vp[i + 32], c = vp[i + 64], d = vp[i + 96];
      a.x = __fmul_rn(a.x, scale); a.y = __fmul_rn(a.y, scale); a.z = __fmul_rn(a.z, scale); a.w = __fmul_rn(a.w, scale);
      b.x = __fmul_rn(b.x, scale); b.y = __fmul_rn(b.y, scale); b.z = __fmul_rn(b.z, scale); b.w = __fmul_rn(b.w, scale);
      c.x = __fmul_rn(c.x, scale); c.y = __fmul_rn(c.y, scale); c.z = __fmul_rn(c.z, scale); c.w = __fmul_rn(c.w, scale);
      d.x = __fmul_rn(d.x, scale); d.y = __fmul_rn(d.y, scale); d.z = __fmul_rn(d.z, scale); d.w = __fmul_rn(d.w, scale);
      vp[i] = a; vp[i + 32] = b; vp[i + 64] = c; vp[i + 96] = d;
    }
    for (; i < nvec; i += 32) {
      float4 a = vp[i];
      a.x = __fmul_rn(a.x, scale); a.y = __fmul_rn(a.y, scale); a.z = __fmul_rn(a.z, scale); a.w = __fmul_rn(a.w, scale);
      vp[i] = a;
    }
    if (tail0 + lane < len) rowp[tail0 + lane] = __fmul_rn(rowp[tail0 + lane], scale);
    if (lane == 0 && scale_out != nullptr) scale_out[row] = scale;
  }
}

int launch_normalize(const rsc_csr& X, float target_sum, const int64_t* cell_total_i64,
                     float* cell_scale_out, cudaStream_t st) {
  if (X.n_rows == 0) return RSC_OK;
  int64_t blocks = (X.n_rows + 7) / 8;
  const int64_t cap = (int64_t)sm_count() * 8;
  if (blocks > cap) blocks = cap;
  normalize_kernel<<<(unsigned)blocks, 256, 0, st>>>(X.n_rows, X.indptr, X.data, target_sum,
                                                     cell_total_i64, cell_scale_out);
  RSC_LAUNCH_CHECK("normalize_kernel");
  return RSC_OK;
}

// ------------------------------------------------------------------ log1p, elementwise
__global__ void __launch_bounds__(256)
log1p_kernel(float* __restrict__ data, int64_t nnz) {
  // 128-bit accesses on the 16-byte aligned body, scalar head/tail.
  const uintptr_t addr = reinterpret_cast<uintptr_t>(data);
  int64_t head = ((16 - (addr & 15)) & 15) >> 2;
  if (head > nnz) head = nnz;
  const int64_t nvec = (nnz - head) >> 2;
  float4* v = reinterpret_cast<float4*>(data + head);
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t nth = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = tid; i < nvec; i += nth) {
    float4 x = v[i];
    x.x = log1p_f32(x.x); x.y = log1p_f32(x.y); x.z = log1p_f32(x.z); x.w = log1p_f32(x.w);
    v[i] = x;
  }
  const int64_t tail0 = head + (nvec << 2);
  if (tid < head) data[tid] = log1p_f32(data[tid]);
  if (tid < nnz - tail0) data[tail0 + tid] = log1p_f32(data[tail0 + tid]);
}

int launch_log1p(const rsc_csr& X, cudaStream_t st) {
  if (X.nnz == 0) return RSC_OK;
  int64_t blocks = (X.nnz / 4 + 255) / 256;
  const int64_t cap = (int64_t)sm_count() * 16;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  log1p_kernel<<<(unsigned)blocks, 256, 0, st>>>(X.data, X.nnz);
  RSC_LAUNCH_CHECK("log1p_kernel");
  return RSC_OK;
}

// ------------------------------------------------------------------ moments, L2 atomics
__global__ void __launch_bounds__(256)
moments_generic_kernel(int64_t nnz, const int32_t* __restrict__ indices,
                       const float* __restrict__ data, int transform, double* __restrict__ S1,
                       double* __restrict__ S2) {
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t nth = (int64_t)gridDim.x * blockDim.x;
  for (int64_t p = tid; p < nnz; p += nth) {
    double v = (double)data[p];
    if (transform == 1) v = expm1(v);
    const int j = indices[p];
    atomicAdd(&S1[j], v);
    atomicAdd(&S2[j], v * v);
  }
}

__global__ void moments_finalize_kernel(int32_t G, double n, double denom,
                                        const double* __restrict__ S1,
                                        const double* __restrict__ S2, double* __restrict__ mean,
                                        double* __restrict__ var) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= G) return;
  const double m = S1[j] / n;
  const double v = (S2[j] - n * m * m) / denom;
  if (mean) mean[j] = m;
  if (var) var[j] = v > 0.0 ? v : (v == v ? 0.0 : v);
}

int finalize_moments(int32_t G, int64_t n, int ddof, const double* S1, const double* S2,
                     double* mean, double* var, cudaStream_t st) {
  moments_finalize_kernel<<<(G + 255) / 256, 256, 0, st>>>(G, (double)n, (double)(n - ddof), S1,
                                                          S2, mean, var);
  RSC_LAUNCH_CHECK("moments_finalize_kernel");
  return RSC_OK;
}

int launch_moments_generic(const rsc_csr& X, int transform, double* S1, double* S2,
                           cudaStream_t st) {
  RSC_CUDA(cudaMemsetAsync(S1, 0, sizeof(double) * X.n_cols, st));
  RSC_CUDA(cudaMemsetAsync(S2, 0, sizeof(double) * X.n_cols, st));
  if (X.nnz == 0) return RSC_OK;
  int64_t blocks = (X.nnz + 255) / 256;
  const int64_t cap = (int64_t)sm_count() * 8;
  if (blocks > cap) blocks = cap;
  moments_generic_kernel<<<(unsigned)blocks, 256, 0, st>>>(X.nnz, X.indices, X.data, transform, S1,
                                                           S2);
  RSC_LAUNCH_CHECK("moments_generic_kernel");
  return RSC_OK;
}

// ------------------------------------------------------------------ fused, warp per row
template <bool LOG, bool LIN>
__global__ void __launch_bounds__(256)
fused_generic_kernel(int64_t n_rows, const int64_t* __restrict__ indptr,
                     const int32_t* __restrict__ indices, float* __restrict__ data,
                     float target_sum, const int64_t* __restrict__ cell_total,
                     double* __restrict__ S1log, double* __restrict__ S2log,
                     double* __restrict__ S1lin, double* __restrict__ S2lin) {
  const int lane = lane_id();
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    const int64_t beg = indptr[row], end = indptr[row + 1];
    const float scale = cell_scale(target_sum, cell_total[row]);
    for (int64_t p = beg + lane; p < end; p += 32) {
      const float xn = __fmul_rn(data[p], scale);
      const float xl = log1p_f32(xn);
      const int j = indices[p];
      data[p] = xl;
      if (LOG) {
        const double v = (double)xl;
        atomicAdd(&S1log[j], v);
        atomicAdd(&S2log[j], v * v);
      }
      if (LIN) {
        const double v = (double)xn;
        atomicAdd(&S1lin[j], v);
        atomicAdd(&S2lin[j], v * v);
      }
    }
  }
}

int launch_fused_generic(const rsc_csr& X, float target_sum, const int64_t* cell_total_i64,
                         int which, double* S1log, double* S2log, double* S1lin, double* S2lin,
                         cudaStream_t st) {
  const size_t gb = sizeof(double) * X.n_cols;
  if (which & RSC_MOMENTS_LOG) {
    RSC_CUDA(cudaMemsetAsync(S1log, 0, gb, st));
    RSC_CUDA(cudaMemsetAsync(S2log, 0, gb, st));
  }
  if (which & RSC_MOMENTS_LIN) {
    RSC_CUDA(cudaMemsetAsync(S1lin, 0, gb, st));
    RSC_CUDA(cudaMemsetAsync(S2lin, 0, gb, st));
  }
  if (X.n_rows == 0) return RSC_OK;
  int64_t blocks = (X.n_rows + 7) / 8;
  const int64_t cap = (int64_t)sm_count() * 8;
  if (blocks > cap) blocks = cap;
  const unsigned b = (unsigned)blocks;
#define RSC_FUSED_ARGS X.n_rows, X.indptr, X.indices, X.data, target_sum, cell_total_i64, S1log, S2log, S1lin, S2lin
  switch (which & 3) {
    case 1: fused_generic_kernel<true, false><<<b, 256, 0, st>>>(RSC_FUSED_ARGS); break;
    case 2: fused_generic_kernel<false, true><<<b, 256, 0, st>>>(RSC_FUSED_ARGS); break;
    case 3: fused_generic_kernel<true, true><<<b, 256, 0, st>>>(RSC_FUSED_ARGS); break;
    default: fused_generic_kernel<false, false><<<b, 256, 0, st>>>(RSC_FUSED_ARGS); break;
  }
#undef RSC_FUSED_ARGS
  RSC_LAUNCH_CHECK("fused_generic_kernel");
  return RSC_OK;
}

}  // namespace rsc
