// Shared host/device helpers of librsc_b200 (CUDA path only; the CPU oracle shares nothing
// with this tree).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <stdio.h>

#include "rsc.h"

namespace rsc {

constexpr int kNumSMs = 148;       // B200: 2 dies x 74 SMs (grid sizing)
constexpr int kWarp = 32;
constexpr size_t kMaxDynSmem = 231424;   // 226 KB dynamic (+ static < 1 KB) <= 227 KB opt-in limit per CTA

// number of column blocks K of the row split table (RSC_SPLIT_WIDTH columns each)
inline int split_blocks(int32_t n_cols) { return (n_cols + RSC_SPLIT_WIDTH - 1) >> RSC_SPLIT_SHIFT; }

void set_error(const char* fmt, ...);

#define RSC_CHECK_ARG(cond, ...)                 \
  do {                                           \
    if (!(cond)) {                               \
      ::rsc::set_error(__VA_ARGS__);             \
      return RSC_ERR_INVALID_ARG;                \
    }                                            \
  } while (0)

#define RSC_CUDA(call)                                                              \
  do {                                                                              \
    cudaError_t e__ = (call);                                                       \
    if (e__ != cudaSuccess) {                                                       \
      ::rsc::set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__),     \
                       __FILE__, __LINE__);                                         \
      return RSC_ERR_CUDA;                                                          \
    }                                                                               \
  } while (0)

// run-time tunables (rsc_set_option): defaults are the shipped configuration
struct Options {                  // process-wide, set through rsc_set_option; atomics: any host thread may set / read
  std::atomic<int> fused_row_budget{256};     // rows a fused-pass CTA takes between two checks of its tables (<= 256)
  std::atomic<int> flush_all{0};              // 1: every check moves every gene to the global totals (testing)
  std::atomic<int> qc_row_budget{512};        // rows a QC CTA takes between two checks of its table (<= 512)
  std::atomic<int> grid_ctas{0};              // CTAs of the streaming kernels; 0 = one per SM
  std::atomic<int> force_generic{0};          // 1: always use the generic L2-atomic kernels
  std::atomic<long long> host_chunk_nnz{150000000};   // rsc_preprocess_host: stored entries per pipelined row chunk
  std::atomic<int> single_pass{0};            // 1: rsc_preprocess takes the one-pass cluster kernel (single.cu) when it can
  std::atomic<int> hvg_single_cta{0};         // 1: rsc_hvg_select on the one-CTA kernel (not the cluster kernel)
};
extern Options g_opt;

extern std::atomic<unsigned long long> g_launch_count;   // kernels launched by this library (host counter)

#define RSC_LAUNCH_CHECK(name)                                                      \
  do {                                                                              \
    ::rsc::g_launch_count.fetch_add(1, std::memory_order_relaxed);                                                      \
    cudaError_t e__ = cudaGetLastError();                                           \
    if (e__ != cudaSuccess) {                                                       \
      ::rsc::set_error("launch of %s failed: %s", name, cudaGetErrorString(e__));   \
      return RSC_ERR_CUDA;                                                          \
    }                                                                               \
  } while (0)

// Returns RSC_OK when the current device is compute capability 10.x.
int check_device();
// Number of SMs of the current device (148 on B200).
int sm_count();

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- launchers implemented in the kernel translation units -------------------------
int launch_qc(const rsc_csr& X, const uint8_t* gene_flags, int64_t* cell_total_i64,
              float* cell_total_f32, int32_t* cell_n_genes, int64_t* cell_flag_total_i64,
              float* cell_flag_pct, int32_t* gene_n_cells, int64_t* gene_total_i64,
              uint32_t* row_splits, const int32_t* split_blocks, int32_t n_split_blocks, void* ws,
              size_t ws_bytes, cudaStream_t st);
// column-block indices at which the fused pass cuts the gene axis (edges of its groups)
int fused_split_blocks(int32_t n_cols, int which, int32_t* out, int32_t cap);
size_t qc_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);
int launch_row_splits(const rsc_csr& X, uint32_t* splits, cudaStream_t st);

int launch_normalize(const rsc_csr& X, float target_sum, const int64_t* cell_total_i64,
                     float* cell_scale_out, cudaStream_t st);
int launch_log1p(const rsc_csr& X, cudaStream_t st);

// mode: 0 = plain moments of data (transform 0/1), 1 = fused normalise+log1p+moments.
int launch_moments(const rsc_csr& X, int transform, int ddof, double* mean, double* var,
                   double* sum, double* sumsq, void* ws, size_t ws_bytes, cudaStream_t st);
size_t moments_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);

int launch_fused(const rsc_csr& X, float target_sum, const int64_t* cell_total_i64,
                 const int32_t* gene_n_cells, const uint32_t* row_splits, int which, int ddof,
                 double* mean_log,
                 double* var_log, double* mean_lin, double* var_lin, double* sums_out, void* ws,
                 size_t ws_bytes, cudaStream_t st);
int finalize_moments(int32_t G, int64_t n, int ddof, const double* S1, const double* S2,
                     double* mean, double* var, cudaStream_t st);
size_t fused_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);

int launch_hvg(int32_t G, const double* mean, const double* var, int32_t n_top, int32_t n_bins,
               int flags, double* out_mean_t, double* out_disp, double* out_disp_norm,
               int32_t* out_bin, uint8_t* out_mask, int32_t* out_indices, int32_t* out_count,
               void* ws, size_t ws_bytes, cudaStream_t st);
size_t hvg_workspace_bytes(int32_t G, int32_t n_bins);

int launch_filter_masks(int64_t n_rows, int32_t n_cols, const int32_t* cell_n_genes,
                        const int64_t* cell_total, const float* cell_pct, const int32_t* gene_n_cells,
                        const int64_t* gene_total, const rsc_filter_params& p, uint8_t* cell_keep,
                        uint8_t* gene_keep, cudaStream_t st);
size_t subset_workspace_bytes(int64_t n_rows, int32_t n_cols);
int launch_subset_plan(const rsc_csr& X, const uint8_t* keep_rows, const uint8_t* keep_cols,
                       int64_t* out_indptr, int64_t* out_counts, void* ws, cudaStream_t st);
int launch_subset_fill(const rsc_csr& X, const uint8_t* keep_rows, int32_t* out_indices, float* out_data,
                       void* ws, cudaStream_t st);

int launch_hvg_cutoffs(int32_t G, const double* mean_t, const double* disp_norm, double min_mean,
                       double max_mean, double min_disp, double max_disp, uint8_t* out_mask,
                       int32_t* out_idx, int32_t* out_count, cudaStream_t st);
size_t scale_workspace_bytes(int32_t n_cols);
int launch_scale_dense(const rsc_csr& X, const double* gene_mean, const double* gene_var,
                       float max_value, int zero_center, float* out, void* ws, cudaStream_t st);

size_t hvg_cell_ranger_workspace_bytes(int32_t G);
int launch_hvg_cell_ranger(int32_t G, const double* mean, const double* var, int32_t n_top, double* out_disp,
                           double* out_disp_norm, int32_t* out_bin, uint8_t* out_mask, int32_t* out_idx,
                           int32_t* out_count, void* ws, cudaStream_t st);
int launch_hvg_merge_batches(int32_t G, int32_t B, const uint8_t* masks, const double* disp_norm, int32_t n_top,
                             int32_t* out_nbatches, double* out_mean, uint8_t* out_mask, int32_t* out_idx,
                             int32_t* out_count, cudaStream_t st);
size_t pca_workspace_bytes(int32_t n_cols, int32_t n_comps);
bool pca_supported(int32_t n_comps);
int launch_pca_transform(const rsc_csr& X, const double* V, const double* mean, int32_t k, float* out, void* ws,
                         cudaStream_t st);
bool single_pass_ok(const rsc_csr& X, int which);
size_t single_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);
int launch_single_pass(const rsc_csr& X, const uint8_t* gene_flags, float target_sum, int ddof,
                       int64_t* cell_total_i64, float* cell_total_f32, int32_t* cell_n_genes,
                       int64_t* cell_flag_total_i64, float* cell_flag_pct, int32_t* gene_n_cells,
                       int64_t* gene_total_i64, double* mean_log, double* var_log, void* ws, cudaStream_t st);
size_t gram_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz);
bool gram_supported(int32_t n_cols);
int launch_gram_cov(const rsc_csr& X, double* out_mean, double* out_gram, double* out_cov, void* ws,
                    size_t ws_bytes, cudaStream_t st);

// ---- device helpers ----------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

template <typename T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Streaming accesses.  The matrix is read once: a line that was used is dead, a line the
// look-ahead has just fetched is not.  Demand loads / stores therefore carry an L2 evict_first
// policy (createpolicy) so that used lines leave the L2 before prefetched ones do.
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ int4 ldg_stream_i4(const void* p, uint64_t pol) {
  int4 v;
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.s32 {%0,%1,%2,%3}, [%4], %5;"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ float4 ldg_stream_f4(const void* p, uint64_t pol) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol));
  return v;
}
// (not .nc: the fused pass rewrites the array it reads)
__device__ __forceinline__ float4 ld_stream_f4(const void* p, uint64_t pol) {
  float4 v;
  asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol) : "memory");
  return v;
}
__device__ __forceinline__ void st_stream_f4(void* p, float4 v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;"
               :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}

// Store of a value this pass will not read again (st.global.cs: evict-first in L2, so the lines the
// look-ahead has fetched stay resident).  Measured per kernel (profiles/r02_cfg3.md): fused pass interior
// quads 3.257 -> 3.185 ms, dense scale output 3.55 -> 3.35 ms; no gain or a loss for normalize, log1p, the
// subset fill and the fused pass's edge quads (their lines are shared with a neighbouring segment that
// another CTA writes later: 3.14 -> 3.31 ms), which keep plain stores.
template <typename T> __device__ __forceinline__ void st_once(T* p, T v) { __stcs(p, v); }

// x'' = log(1 + x') in float32, shared by rsc_log1p and the fused pass so that
// both write bit-identical values.  x >= 0.25: MUFU lg2 of the rounded 1 + x (absolute error
// <= 2^-22 * ln 2 + 2^-24, i.e. <= 1e-6 relative there, ~1 ulp for typical x'' of 1..3);
// |x| < 0.25: x * (1 - x/2 + x^2/3 - ... - x^9/10), truncation < 1e-7 relative.
// The stated tolerance on x'' is 1e-5 relative (north_star).
__device__ __forceinline__ float log1p_ge_quarter(float x) {      // x >= 0.25 (1 + x is normal)
  float l;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"(__fadd_rn(1.0f, x)));
  return __fmul_rn(l, 0.693147182f);
}
__device__ __forceinline__ float log1p_f32(float x) {
  if (x >= 0.25f) return log1p_ge_quarter(x);
  if (x < -0.25f) return log1pf(x);
  float p = -0.1f;
  p = fmaf(p, x, 1.0f / 9.0f);
  p = fmaf(p, x, -0.125f);
  p = fmaf(p, x, 1.0f / 7.0f);
  p = fmaf(p, x, -1.0f / 6.0f);
  p = fmaf(p, x, 0.2f);
  p = fmaf(p, x, -0.25f);
  p = fmaf(p, x, 1.0f / 3.0f);
  p = fmaf(p, x, -0.5f);
  p = fmaf(p, x, 1.0f);
  return x * p;
}

// scale_i of normalize_total: one float32 division, shared by the unfused and the fused
// kernels so that their x' are bit-identical (reading R5).
__device__ __forceinline__ float cell_scale(float target_sum, int64_t total) {
  return total != 0 ? __fdiv_rn(target_sum, (float)total) : 1.0f;
}
#endif

}  // namespace rsc
