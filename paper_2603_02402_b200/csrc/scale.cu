// SURVEY.md 8(f) NEXT-3 (first half): scale -- z-score per gene with optional clip ("scaling",
// PAPER.md:L61, L151), from the per-gene mean / variance the preprocessing chain already produced.
// The output is DENSE float32 [n_rows, n_cols] (the step densifies; it follows HVG subsetting):
//     y_ij = clip((x_ij - mean_j) / sd_j),  sd_j = sqrt(var_j), 1 where var_j == 0
// Every row is first filled with the per-gene value of a zero entry (one 128-bit store per lane,
// from a small table), then the row's stored entries overwrite their positions; the entries are
// computed in fp64 (no cancellation error near the mean).  Write-bound: 4 B x n_rows x n_cols.
#include <math.h>

#include "common.cuh"

namespace rsc {

// per-gene 1 / sd (double; sd = 1 where the variance is 0) and the value of a zero entry (float, clipped)
__global__ void __launch_bounds__(256)
scale_prep_kernel(int32_t G, const double* __restrict__ mean, const double* __restrict__ var,
                  float max_value, int zero_center, double* __restrict__ inv_sd_out, float* __restrict__ base) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= G) return;
  double sd = sqrt(var[j]);
  if (sd == 0.0) sd = 1.0;
  const double inv = 1.0 / sd;
  inv_sd_out[j] = inv;                                         // the entries multiply by 1 / sd (one rounding more than
                                                           // the definition's division, in double: far below float32)
  double b = zero_center ? (0.0 - mean[j]) * inv : 0.0;
  if (max_value > 0.0f) {
    if (b > (double)max_value) b = (double)max_value;
    if (zero_center && b < -(double)max_value) b = -(double)max_value;
  }
  base[j] = (float)b;
}

__global__ void __launch_bounds__(256)
scale_dense_kernel(int64_t n_rows, int32_t G, const int64_t* __restrict__ indptr,
                   const int32_t* __restrict__ indices, const float* __restrict__ data,
                   const double* __restrict__ mean, const double* __restrict__ inv_sd,
                   const float* __restrict__ base, float max_value, int zero_center,
                   float* __restrict__ out) {
  const int lane = lane_id();
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const bool vec = (G & 3) == 0 && ((reinterpret_cast<uintptr_t>(out) | reinterpret_cast<uintptr_t>(base)) & 15) == 0;
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    float* o = out + row * (int64_t)G;
    if (vec) {
      for (int j = lane * 4; j < G; j += 128)
        *reinterpret_cast<float4*>(o + j) = __ldg(reinterpret_cast<const float4*>(base + j));
    } else {
      for (int j = lane; j < G; j += 32) o[j] = __ldg(base + j);
    }
    __syncwarp();                                          // the fill is ordered before the overwrites
    const int64_t beg = indptr[row], end = indptr[row + 1];
    for (int64_t p = beg + lane; p < end; p += 32) {
      const int j = __ldg(indices + p);
      double y = (double)__ldg(data + p);
      if (zero_center) y -= mean[j];
      y = y * inv_sd[j];
      if (max_value > 0.0f) {
        if (y > (double)max_value) y = (double)max_value;
        if (zero_center && y < -(double)max_value) y = -(double)max_value;
      }
      o[j] = (float)y;
    }
  }
}

// The same with the row staged in shared memory (G % 4 == 0, 4 rows of G floats per CTA fit):
// the row is assembled on chip and leaves the SM once, as full 128-bit stores -- the scattered
// 4-byte overwrites of the direct kernel cost more than its whole fill phase (measured).
constexpr int kScaleWarps = 4;
__global__ void __launch_bounds__(kScaleWarps * 32)
scale_dense_smem_kernel(int64_t n_rows, int32_t G, const int64_t* __restrict__ indptr,
                        const int32_t* __restrict__ indices, const float* __restrict__ data,
                        const double* __restrict__ mean, const double* __restrict__ inv_sd,
                        const float* __restrict__ base, float max_value, int zero_center,
                        float* __restrict__ out) {
  extern __shared__ __align__(16) float srow[];
  const int lane = lane_id(), warp = threadIdx.x >> 5;
  float* r = srow + (size_t)warp * G;
  const int64_t warp0 = (int64_t)blockIdx.x * kScaleWarps + warp;
  const int64_t nwarps = (int64_t)gridDim.x * kScaleWarps;
  auto zscore = [&](int j, float x) -> float {
    double y = (double)x;
    if (zero_center) y -= mean[j];
    y = y * inv_sd[j];
    if (max_value > 0.0f) {
      if (y > (double)max_value) y = (double)max_value;
      if (zero_center && y < -(double)max_value) y = -(double)max_value;
    }
    return (float)y;
  };
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    // the row's first 128 entries are requested before the fill, whose stores hide their latency;
    // the next row of this warp goes to L2
    const int64_t beg = indptr[row], end = indptr[row + 1];
    int j4[4];
    float x4[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t p = beg + u * 32 + lane;
      j4[u] = p < end ? __ldg(indices + p) : -1;
      x4[u] = p < end ? __ldg(data + p) : 0.0f;
    }
    if (row + nwarps < n_rows) {
      const int64_t nb = indptr[row + nwarps], ne = indptr[row + nwarps + 1];
      for (int64_t p = (nb & ~31LL) + lane * 32; p < ne; p += 32 * 32) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(indices + p));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(data + p));
      }
    }
    for (int j = lane * 4; j < G; j += 128)
      *reinterpret_cast<float4*>(r + j) = __ldg(reinterpret_cast<const float4*>(base + j));
    __syncwarp();
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (j4[u] >= 0) r[j4[u]] = zscore(j4[u], x4[u]);
    for (int64_t p = beg + 128 + lane; p < end; p += 32) {
      const int j = __ldg(indices + p);
      r[j] = zscore(j, __ldg(data + p));
    }
    __syncwarp();
    float* o = out + row * (int64_t)G;
    for (int j = lane * 4; j < G; j += 128)
      *reinterpret_cast<float4*>(o + j) = *reinterpret_cast<const float4*>(r + j);
    __syncwarp();
  }
}

// Sorted rows: the row is produced in column chunks of kScaleChunk genes, so a warp stages only
// 4 KB (not the whole row) and many more warps fit an SM.  The values of zero entries come from a
// CTA-wide copy of the table in shared memory (read from L2 once per CTA, not once per row).  The
// entries of a chunk are a contiguous run of the sorted row: the warp keeps a batch of 32 entries
// in registers (one coalesced load per array), scatters the ones that fall into the current chunk
// and refills the batch when all of it has been used.  Per chunk: fill, scatter, one 128-bit
// store per lane and 128 genes: the output is written exactly once, as full lines.
// (Measured slower: handing the entries to their owner lanes by shuffles and storing straight
// from registers, 7.1 ms -- one serial shuffle round per entry.)
#ifndef RSC_SC_CHUNK
#define RSC_SC_CHUNK 1024
#endif
#ifndef RSC_SC_WARPS
#define RSC_SC_WARPS 8
#endif
constexpr int kScaleChunk = RSC_SC_CHUNK;
constexpr int kScaleChunkWarps = RSC_SC_WARPS;
__global__ void __launch_bounds__(kScaleChunkWarps * 32)
scale_dense_chunk_kernel(int64_t n_rows, int32_t G, const int64_t* __restrict__ indptr,
                         const int32_t* __restrict__ indices, const float* __restrict__ data,
                         const double2* __restrict__ mean_inv, const float* __restrict__ base,
                         float max_value, int zero_center, float* __restrict__ out) {
  extern __shared__ __align__(16) float ssm[];             // [warps][kScaleChunk] staging | [G] zero-entry values
  const int lane = lane_id(), warp = threadIdx.x >> 5;
  float* r = ssm + warp * kScaleChunk;
  float* sbase = ssm + kScaleChunkWarps * kScaleChunk;
  for (int t = threadIdx.x * 4; t < G; t += kScaleChunkWarps * 32 * 4)
    *reinterpret_cast<float4*>(sbase + t) = __ldg(reinterpret_cast<const float4*>(base + t));
  __syncthreads();
  const int64_t warp0 = (int64_t)blockIdx.x * kScaleChunkWarps + warp;
  const int64_t nwarps = (int64_t)gridDim.x * kScaleChunkWarps;
  constexpr int kNone = 0x7fffffff;
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    const int64_t beg = indptr[row], end = indptr[row + 1];
    int64_t p = beg;                                       // first entry of the batch in registers
    int j = kNone;
    float y = 0.0f;
    auto load_batch = [&]() {
      j = kNone;
      if (p + lane < end) {
        j = __ldg(indices + p + lane);
        const double2 mi = __ldg(mean_inv + j);
        double v = (double)__ldg(data + p + lane);
        if (zero_center) v -= mi.x;
        v *= mi.y;
        if (max_value > 0.0f) {
          if (v > (double)max_value) v = (double)max_value;
          if (zero_center && v < -(double)max_value) v = -(double)max_value;
        }
        y = (float)v;
      }
    };
    load_batch();
    if (row + nwarps < n_rows) {                           // the warp's next row goes to L2
      const int64_t nb = indptr[row + nwarps], ne = indptr[row + nwarps + 1];
      for (int64_t q = (nb & ~31LL) + lane * 32; q < ne; q += 32 * 32) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(indices + q));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(data + q));
      }
    }
    float* o = out + row * (int64_t)G;
    for (int c0 = 0; c0 < G; c0 += kScaleChunk) {
      const int c1 = min(G, c0 + kScaleChunk);
      for (int t = lane * 4; t < c1 - c0; t += 128)
        *reinterpret_cast<float4*>(r + t) = *reinterpret_cast<const float4*>(sbase + c0 + t);
      __syncwarp();
      for (;;) {
        if (j < c1) { r[j - c0] = y; j = kNone; }          // (j >= c0: earlier chunks consumed theirs)
        if (__all_sync(0xffffffffu, j == kNone) && p + 32 < end) { p += 32; load_batch(); }
        else break;
      }
      __syncwarp();
      for (int t = lane * 4; t < c1 - c0; t += 128)
        st_once(reinterpret_cast<float4*>(o + c0 + t), *reinterpret_cast<const float4*>(r + t));
      __syncwarp();
    }
  }
}

__global__ void __launch_bounds__(256)
scale_pack_table_kernel(int32_t G, const double* __restrict__ mean, const double* __restrict__ inv_sd,
                        double2* __restrict__ mean_inv) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < G) mean_inv[j] = make_double2(mean[j], inv_sd[j]);
}

size_t scale_workspace_bytes(int32_t n_cols) {
  return align_up(sizeof(double) * (size_t)(n_cols > 0 ? n_cols : 0), 256) +
         align_up(sizeof(float) * (size_t)(n_cols > 0 ? n_cols : 0), 256) +
         align_up(sizeof(double2) * (size_t)(n_cols > 0 ? n_cols : 0), 256);
}

int launch_scale_dense(const rsc_csr& X, const double* gene_mean, const double* gene_var,
                       float max_value, int zero_center, float* out, void* ws, cudaStream_t st) {
  if (X.n_rows == 0) return RSC_OK;
  unsigned char* w = static_cast<unsigned char*>(ws);
  double* inv_sd = reinterpret_cast<double*>(w);
  float* base = reinterpret_cast<float*>(w + align_up(sizeof(double) * (size_t)X.n_cols, 256));
  scale_prep_kernel<<<(X.n_cols + 255) / 256, 256, 0, st>>>(X.n_cols, gene_mean, gene_var, max_value,
                                                            zero_center, inv_sd, base);
  RSC_LAUNCH_CHECK("scale_prep_kernel");
  const bool aligned16 = ((reinterpret_cast<uintptr_t>(out) | reinterpret_cast<uintptr_t>(base)) & 15) == 0;
  if ((X.flags & RSC_CSR_SORTED) && (X.n_cols & 3) == 0 && aligned16 && !g_opt.force_generic &&
      sizeof(float) * ((size_t)X.n_cols + (size_t)kScaleChunkWarps * kScaleChunk) <= 220 * 1024) {
    double2* mean_inv = reinterpret_cast<double2*>(w + align_up(sizeof(double) * (size_t)X.n_cols, 256) +
                                                   align_up(sizeof(float) * (size_t)X.n_cols, 256));
    scale_pack_table_kernel<<<(X.n_cols + 255) / 256, 256, 0, st>>>(X.n_cols, gene_mean, inv_sd, mean_inv);
    RSC_LAUNCH_CHECK("scale_pack_table_kernel");
    const size_t bsm = sizeof(float) * ((size_t)X.n_cols + (size_t)kScaleChunkWarps * kScaleChunk);
    RSC_CUDA(cudaFuncSetAttribute(scale_dense_chunk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsm));
    int per_sm = (int)((220 * 1024) / (bsm + 1024));
    per_sm = per_sm > 6 ? 6 : (per_sm < 1 ? 1 : per_sm);
    int64_t blocks = (X.n_rows + kScaleChunkWarps - 1) / kScaleChunkWarps;
    const int64_t cap = (int64_t)sm_count() * per_sm;
    if (blocks > cap) blocks = cap;
    scale_dense_chunk_kernel<<<(unsigned)blocks, kScaleChunkWarps * 32, bsm, st>>>(
        X.n_rows, X.n_cols, X.indptr, X.indices, X.data, mean_inv, base, max_value, zero_center, out);
    RSC_LAUNCH_CHECK("scale_dense_chunk_kernel");
    return RSC_OK;
  }
  const size_t smem = sizeof(float) * (size_t)kScaleWarps * (size_t)X.n_cols;
  const bool staged = (X.n_cols & 3) == 0 && smem <= 100 * 1024 &&
                      ((reinterpret_cast<uintptr_t>(out) | reinterpret_cast<uintptr_t>(base)) & 15) == 0;
  if (staged) {
    RSC_CUDA(cudaFuncSetAttribute(scale_dense_smem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)(100 * 1024)));
    const int per_sm = (int)((220 * 1024) / (smem + 1024)) > 0 ? (int)((220 * 1024) / (smem + 1024)) : 1;
    int64_t blocks = (X.n_rows + kScaleWarps - 1) / kScaleWarps;
    const int64_t cap = (int64_t)sm_count() * (per_sm > 16 ? 16 : per_sm);
    if (blocks > cap) blocks = cap;
    scale_dense_smem_kernel<<<(unsigned)blocks, kScaleWarps * 32, smem, st>>>(
        X.n_rows, X.n_cols, X.indptr, X.indices, X.data, gene_mean, inv_sd, base, max_value, zero_center, out);
    RSC_LAUNCH_CHECK("scale_dense_smem_kernel");
    return RSC_OK;
  }
  int64_t blocks = (X.n_rows + 7) / 8;
  const int64_t cap = (int64_t)sm_count() * 16;
  if (blocks > cap) blocks = cap;
  scale_dense_kernel<<<(unsigned)blocks, 256, 0, st>>>(X.n_rows, X.n_cols, X.indptr, X.indices, X.data,
                                                       gene_mean, inv_sd, base, max_value, zero_center, out);
  RSC_LAUNCH_CHECK("scale_dense_kernel");
  return RSC_OK;
}

}  // namespace rsc
