// Device-side Seurat-flavour HVG selection: dispersion transform, equal-width mean bins,
// per-bin z-score, exact top-k by radix select, ordered compaction.  One CTA: the problem
// is G <= ~36 k doubles ("gene selection" kernel avoiding CPU<->GPU
// transfers; L91 "based on per-gene mean and variance").  Steps H1..H7 of DESIGN.md §3.
#include <math.h>

#include "common.cuh"

namespace rsc {

constexpr int kHvgThreads = 1024;
constexpr int kHvgWarps = kHvgThreads / 32;

__device__ __forceinline__ unsigned long long z_key(double z) {
  // order-preserving map double -> uint64 (larger z <=> larger key); -0.0 canonicalised
  z = z + 0.0;
  const unsigned long long b = (unsigned long long)__double_as_longlong(z);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}

__global__ void __launch_bounds__(kHvgThreads)
hvg_kernel(int G, const double* __restrict__ mean, const double* __restrict__ var, int n_top,
           int n_bins, int flags, double* __restrict__ m_arr, double* __restrict__ d_arr,
           double* __restrict__ z_arr, int32_t* __restrict__ bin_arr,
           uint8_t* __restrict__ out_mask, int32_t* __restrict__ out_idx,
           int32_t* __restrict__ out_count) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* edges = reinterpret_cast<double*>(smem_raw);         // n_bins + 1
  double* mu_b = edges + (n_bins + 1);                         // n_bins
  double* sd_b = mu_b + n_bins;                                // n_bins
  double* red = sd_b + n_bins;                                 // 2 * kHvgWarps
  int* hist = reinterpret_cast<int*>(red + 2 * kHvgWarps);     // 256
  int* wsum = hist + 256;                                      // kHvgWarps
  __shared__ unsigned long long s_prefix;
  __shared__ int s_remaining, s_nvalid, s_base;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const double kNaN = __longlong_as_double(0x7ff8000000000000ll);

  // H1 / H2: dispersion and transforms; min / max of the transformed mean
  double lo = __longlong_as_double(0x7ff0000000000000ll), hi = -lo;
  for (int g = tid; g < G; g += kHvgThreads) {
    double mu = mean[g];
    if (mu == 0.0) mu = 1e-12;
    double d = __ddiv_rn(var[g], mu);
    double m = mu;
    if (flags & RSC_HVG_SEURAT_LOG) {
      if (d == 0.0) d = kNaN;
      d = log(d);
      m = log1p(mu);
    }
    m_arr[g] = m;
    d_arr[g] = d;
    lo = fmin(lo, m);
    hi = fmax(hi, m);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if (lane == 0) { red[warp] = lo; red[kHvgWarps + warp] = hi; }
  __syncthreads();
  lo = red[0]; hi = red[kHvgWarps];
  for (int w = 1; w < kHvgWarps; ++w) { lo = fmin(lo, red[w]); hi = fmax(hi, red[kHvgWarps + w]); }

  // H3: edges, separate multiply and add (no FMA contraction) to match numpy.linspace
  const bool degenerate = (lo == hi);
  if (degenerate) {
    lo = __dsub_rn(lo, lo != 0.0 ? __dmul_rn(0.001, fabs(lo)) : 0.001);
    hi = __dadd_rn(hi, hi != 0.0 ? __dmul_rn(0.001, fabs(hi)) : 0.001);
  }
  const double step = __ddiv_rn(__dsub_rn(hi, lo), (double)n_bins);
  for (int k = tid; k <= n_bins; k += kHvgThreads) {
    double e = (k == n_bins) ? hi : __dadd_rn(__dmul_rn((double)k, step), lo);
    if (k == 0 && !degenerate) e = __dsub_rn(e, __dmul_rn(__dsub_rn(hi, lo), 0.001));
    edges[k] = e;
  }
  __syncthreads();

  // H4: bin(m) = smallest k with m <= edge_{k+1}
  for (int g = tid; g < G; g += kHvgThreads) {
    const double m = m_arr[g];
    int a = 0, b = n_bins - 1;
    while (a < b) {
      const int mid = (a + b) >> 1;
      if (m <= edges[mid + 1]) b = mid; else a = mid + 1;
    }
    bin_arr[g] = a;
  }
  __syncthreads();

  // H5: per-bin mean and sample sd of the non-NaN dispersions (two passes, one warp per bin)
  for (int b = warp; b < n_bins; b += kHvgWarps) {
    double s = 0.0;
    int c = 0;
    for (int g = lane; g < G; g += 32) {
      if (bin_arr[g] == b) {
        const double d = d_arr[g];
        if (d == d) { s += d; ++c; }
      }
    }
    s = warp_sum(s);
    c = warp_sum(c);
    const double mk = s / (double)c;
    double ss = 0.0;
    for (int g = lane; g < G; g += 32) {
      if (bin_arr[g] == b) {
        const double d = d_arr[g];
        if (d == d) { const double t = d - mk; ss += t * t; }
      }
    }
    ss = warp_sum(ss);
    if (lane == 0) {
      if (c == 0) { mu_b[b] = kNaN; sd_b[b] = kNaN; }
      else if (c == 1) { mu_b[b] = 0.0; sd_b[b] = mk; }
      else { mu_b[b] = mk; sd_b[b] = sqrt(ss / (double)(c - 1)); }
    }
  }
  if (tid == 0) { s_prefix = 0ull; s_nvalid = 0; }
  __syncthreads();

  // H6: z-score; count the valid (non-NaN) genes
  int nv = 0;
  for (int g = tid; g < G; g += kHvgThreads) {
    const int b = bin_arr[g];
    const double z = __ddiv_rn(__dsub_rn(d_arr[g], mu_b[b]), sd_b[b]);
    z_arr[g] = z;
    nv += (z == z);
  }
  nv = warp_sum(nv);
  if (lane == 0 && nv) atomicAdd(&s_nvalid, nv);
  __syncthreads();
  const int k_sel = min(n_top, s_nvalid);

  // H7: exact k-th largest by 8 x 8-bit radix select on the order-preserving keys
  if (k_sel > 0) {
    if (tid == 0) s_remaining = k_sel;
    unsigned long long have_mask = 0ull;
    for (int pass = 7; pass >= 0; --pass) {
      const int shift = pass * 8;
      for (int i = tid; i < 256; i += kHvgThreads) hist[i] = 0;
      __syncthreads();
      const unsigned long long prefix = s_prefix;
      for (int g = tid; g < G; g += kHvgThreads) {
        const double z = z_arr[g];
        if (z == z) {
          const unsigned long long key = z_key(z);
          if ((key & have_mask) == prefix) atomicAdd(&hist[(int)((key >> shift) & 255ull)], 1);
        }
      }
      __syncthreads();
      if (tid == 0) {
        int rem = s_remaining, dgt = 255;
        for (; dgt > 0; --dgt) {
          if (hist[dgt] >= rem) break;
          rem -= hist[dgt];
        }
        s_remaining = rem;
        s_prefix = prefix | ((unsigned long long)dgt << shift);
      }
      have_mask |= (255ull << shift);
      __syncthreads();
    }
  }
  const unsigned long long cut = s_prefix;
  if (tid == 0) s_base = 0;
  __syncthreads();

  // mask + ascending index list (ordered block compaction, 1024 genes per round)
  for (int g0 = 0; g0 < G; g0 += kHvgThreads) {
    const int g = g0 + tid;
    bool sel = false;
    if (g < G && k_sel > 0) {
      const double z = z_arr[g];
      sel = (z == z) && (z_key(z) >= cut);
    }
    if (g < G) out_mask[g] = sel ? 1 : 0;
    const unsigned bal = __ballot_sync(0xffffffffu, sel);
    if (lane == 0) wsum[warp] = __popc(bal);
    __syncthreads();
    int off = s_base;
    for (int w = 0; w < warp; ++w) off += wsum[w];
    if (sel && out_idx != nullptr) out_idx[off + __popc(bal & ((1u << lane) - 1u))] = g;
    __syncthreads();
    if (tid == 0) {
      int t = s_base;
      for (int w = 0; w < kHvgWarps; ++w) t += wsum[w];
      s_base = t;
    }
    __syncthreads();
  }
  if (tid == 0) *out_count = s_base;
}

size_t hvg_workspace_bytes(int32_t G, int32_t /*n_bins*/) {
  // m, d, z (double) + bin (int32), each 256-byte aligned
  return 3 * align_up(sizeof(double) * (size_t)G, 256) + align_up(sizeof(int32_t) * (size_t)G, 256);
}

int launch_hvg(int32_t G, const double* mean, const double* var, int32_t n_top, int32_t n_bins,
               int flags, double* out_mean_t, double* out_disp, double* out_disp_norm,
               int32_t* out_bin, uint8_t* out_mask, int32_t* out_indices, int32_t* out_count,
               void* ws, size_t ws_bytes, cudaStream_t st) {
  if (ws_bytes < hvg_workspace_bytes(G, n_bins) || ws == nullptr ||
      (reinterpret_cast<uintptr_t>(ws) & 255)) {
    set_error("rsc_hvg_select: workspace too small or misaligned (%zu < %zu)", ws_bytes,
              hvg_workspace_bytes(G, n_bins));
    return RSC_ERR_WORKSPACE;
  }
  unsigned char* w = static_cast<unsigned char*>(ws);
  const size_t dsz = align_up(sizeof(double) * (size_t)G, 256);
  double* m_arr = out_mean_t ? out_mean_t : reinterpret_cast<double*>(w);
  double* d_arr = out_disp ? out_disp : reinterpret_cast<double*>(w + dsz);
  double* z_arr = out_disp_norm ? out_disp_norm : reinterpret_cast<double*>(w + 2 * dsz);
  int32_t* b_arr = out_bin ? out_bin : reinterpret_cast<int32_t*>(w + 3 * dsz);
  const size_t smem = sizeof(double) * (3 * (size_t)n_bins + 1 + 2 * kHvgWarps) +
                      sizeof(int) * (256 + kHvgWarps);
  if (smem > 48 * 1024) {
    RSC_CUDA(cudaFuncSetAttribute(hvg_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)smem));
  }
  hvg_kernel<<<1, kHvgThreads, smem, st>>>(G, mean, var, n_top, n_bins, flags, m_arr, d_arr, z_arr,
                                           b_arr, out_mask, out_indices, out_count);
  RSC_LAUNCH_CHECK("hvg_kernel");
  return RSC_OK;
}

}  // namespace rsc
