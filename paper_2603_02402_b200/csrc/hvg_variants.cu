// the other HVG variants on the device ("Highly variable gene
// selection is based on per-gene mean and variance", L39 "gene selection" without CPU round trips,
// L87 "follow the algorithmic implementations of scanpy"; the constants are not in the paper:
// DESIGN.md readings R18 / R19).
//   * rsc_hvg_select_cell_ranger: percentile bins of the mean (P10, P15, .., P100), dispersion
//     normalised by the bin's median and MAD, top-k by the normalised dispersion;
//   * rsc_hvg_merge_batches: per-batch selections merged by (number of batches, mean normalised
//     dispersion).
// G <= 57 k values: one CTA.  Every order statistic (percentile, median, MAD, cutoff) is an EXACT
// selection: one warp runs an 8 x 8-bit most-significant-digit radix select over order-preserving
// 64-bit keys (shared-memory histogram per warp), several warps serve several bins / percentiles
// at once.  No sorting, no floating-point histogram edges: the results equal the oracle's bit for
// bit wherever it takes an element of the data (edges, medians use the same separate multiply / add).
#include <math.h>

#include "common.cuh"

namespace rsc {

constexpr int kHv2Threads = 1024;
constexpr int kHv2Warps = kHv2Threads / 32;
constexpr int kCrMaxEdges = 21;              // -inf, P10 .. P100, +inf
constexpr double kMadScale = 0.6744897501960817;

// ascending order-preserving key of a non-NaN double
__device__ __forceinline__ unsigned long long dkey(double v) {
  const unsigned long long b = (unsigned long long)__double_as_longlong(v);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double dkey_inv(unsigned long long k) {
  const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
  return __longlong_as_double((long long)b);
}

// k-th smallest (k = 1 .. count) key among the items i in [0, n) for which f(i, key) is true.
// One warp; hist = 256 ints of shared memory owned by this warp.  The caller guarantees
// 1 <= k <= number of accepted items.
template <typename F>
__device__ unsigned long long warp_select(int n, int k, int* hist, F f) {
  const int lane = threadIdx.x & 31;
  unsigned long long prefix = 0ull;                       // the digits fixed so far (high bits)
  for (int pass = 7; pass >= 0; --pass) {
    for (int i = lane; i < 256; i += 32) hist[i] = 0;
    __syncwarp();
    const int sh = pass * 8;
    for (int i = lane; i < n; i += 32) {
      unsigned long long key;
      if (f(i, key) && (pass == 7 || (key >> (sh + 8)) == prefix)) atomicAdd(&hist[(int)((key >> sh) & 255ull)], 1);
    }
    __syncwarp();
    // lane l owns digits 8 l .. 8 l + 7
    int c[8], s = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { c[j] = hist[lane * 8 + j]; s += c[j]; }
    int incl = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    int below = incl - s;                                 // items in digits of the lanes before me
    int digit = -1, kk = 0;
    if (k > below && k <= incl) {                         // exactly one lane
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (digit < 0 && k <= below + c[j]) { digit = lane * 8 + j; kk = k - below; }
        if (digit < 0) below += c[j];
      }
    }
    const unsigned who = __ballot_sync(0xffffffffu, digit >= 0);
    const int src = __ffs(who) - 1;
    digit = __shfl_sync(0xffffffffu, digit, src);
    k = __shfl_sync(0xffffffffu, kk, src);
    prefix = (prefix << 8) | (unsigned long long)digit;
    __syncwarp();
  }
  return prefix;
}

// ordered compaction of the selected genes (ascending) + count; every thread owns a contiguous chunk
__device__ void cta_compact(int G, const uint8_t* __restrict__ mask, int32_t* __restrict__ out_idx,
                            int32_t* __restrict__ out_count, int* scan /* kHv2Threads + 1 ints */) {
  const int tid = threadIdx.x;
  const int per = (G + kHv2Threads - 1) / kHv2Threads;
  const int g0 = min(G, tid * per), g1 = min(G, g0 + per);
  int c = 0;
  for (int g = g0; g < g1; ++g) c += mask[g] ? 1 : 0;
  scan[tid + 1] = c;
  if (tid == 0) scan[0] = 0;
  __syncthreads();
  if (tid < 32) {                                         // one warp scans the 1024 counts
    int carry = 0;
    for (int b = 0; b < kHv2Threads; b += 32) {
      const int v = scan[b + tid + 1];
      int incl = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (tid >= o) incl += t;
      }
      scan[b + tid + 1] = carry + incl;
      carry += __shfl_sync(0xffffffffu, incl, 31);
    }
  }
  __syncthreads();
  if (out_idx != nullptr) {
    int o = scan[tid];
    for (int g = g0; g < g1; ++g)
      if (mask[g]) out_idx[o++] = g;
  }
  if (tid == 0) out_count[0] = scan[kHv2Threads];
}

// ------------------------------------------------------------------ cell-ranger flavour
__global__ void __launch_bounds__(kHv2Threads)
hvg_cell_ranger_kernel(int G, const double* __restrict__ mean, const double* __restrict__ var, int n_top,
                       double* __restrict__ d_arr, double* __restrict__ z_arr, int32_t* __restrict__ bin_arr,
                       uint8_t* __restrict__ out_mask, int32_t* __restrict__ out_idx,
                       int32_t* __restrict__ out_count) {
  __shared__ int hist[kHv2Warps][256];
  __shared__ int scan[kHv2Threads + 1];
  __shared__ double pct[kCrMaxEdges], edges[kCrMaxEdges + 1], med[kCrMaxEdges], mad[kCrMaxEdges];
  __shared__ int s_nb, s_nvalid;
  __shared__ double s_cut;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const double kNaN = __longlong_as_double(0x7ff8000000000000ll);
  const double kInf = __longlong_as_double(0x7ff0000000000000ll);

  // C1: dispersion (mean == 0 -> 1e-12)
  for (int g = tid; g < G; g += kHv2Threads) {
    const double m = mean[g];
    d_arr[g] = __ddiv_rn(var[g], m == 0.0 ? 1e-12 : m);
  }
  if (tid == 0) s_nvalid = 0;
  // C2: P10, P15, .., P100 of the means: warp w takes percentile 10 + 5 w (linear interpolation
  // between two exact order statistics; separate multiply / add, as oracle_np.percentile_linear)
  if (warp < 19) {
    const double q = (double)(10 + 5 * warp);
    const double vi = __dmul_rn(__ddiv_rn(q, 100.0), (double)(G - 1));
    const int lo = (int)floor(vi);
    const int hi = min(lo + 1, G - 1);
    const double t = __dsub_rn(vi, (double)lo);
    auto key_of = [&](int i, unsigned long long& key) -> bool { key = dkey(mean[i]); return true; };
    const double a = dkey_inv(warp_select(G, lo + 1, hist[warp], key_of));
    const double b = hi == lo ? a : dkey_inv(warp_select(G, hi + 1, hist[warp], key_of));
    const double diff = __dsub_rn(b, a);
    const double v = t < 0.5 ? __dadd_rn(a, __dmul_rn(diff, t)) : __dsub_rn(b, __dmul_rn(diff, __dsub_rn(1.0, t)));
    if (lane == 0) pct[warp] = v;
  }
  __syncthreads();
  if (tid == 0) {                                         // merged edges (equal edges collapse)
    int ne = 0;
    edges[ne++] = -kInf;
    for (int k = 0; k < 19; ++k)
      if (pct[k] != edges[ne - 1]) edges[ne++] = pct[k];
    if (kInf != edges[ne - 1]) edges[ne++] = kInf;
    s_nb = ne - 1;
  }
  __syncthreads();
  const int nb = s_nb;
  // C3: bin(m) = smallest k with m <= e_{k+1}
  for (int g = tid; g < G; g += kHv2Threads) {
    const double m = mean[g];
    int k = 0;
    while (k < nb - 1 && !(m <= edges[k + 1])) ++k;
    bin_arr[g] = k;
  }
  __syncthreads();
  // C4: per bin (one warp each): median of d, then MAD = median |d - med| / 0.6745
  for (int b = warp; b < nb; b += kHv2Warps) {
    int c = 0;
    for (int g = lane; g < G; g += 32) {
      const double d = d_arr[g];
      c += (bin_arr[g] == b && d == d) ? 1 : 0;
    }
    c = warp_sum(c);
    double mb = kNaN, ab = kNaN;
    if (c > 0) {
      const int k1 = (c - 1) / 2 + 1, k2 = c / 2 + 1;      // 1-based ranks of the two middle values
      auto key_d = [&](int i, unsigned long long& key) -> bool {
        const double d = d_arr[i];
        key = dkey(d);
        return bin_arr[i] == b && d == d;
      };
      const double v1 = dkey_inv(warp_select(G, k1, hist[warp], key_d));
      const double v2 = k2 == k1 ? v1 : dkey_inv(warp_select(G, k2, hist[warp], key_d));
      mb = __dmul_rn(__dadd_rn(v1, v2), 0.5);
      auto key_a = [&](int i, unsigned long long& key) -> bool {
        const double d = d_arr[i];
        key = dkey(fabs(__dsub_rn(d, mb)));
        return bin_arr[i] == b && d == d;
      };
      const double a1 = dkey_inv(warp_select(G, k1, hist[warp], key_a));
      const double a2 = k2 == k1 ? a1 : dkey_inv(warp_select(G, k2, hist[warp], key_a));
      ab = __ddiv_rn(__dmul_rn(__dadd_rn(a1, a2), 0.5), kMadScale);
    }
    if (lane == 0) { med[b] = mb; mad[b] = ab; }
  }
  __syncthreads();
  // C5: z = (d - med) / mad; count the non-NaN z
  int nv = 0;
  for (int g = tid; g < G; g += kHv2Threads) {
    const int b = bin_arr[g];
    const double z = __ddiv_rn(__dsub_rn(d_arr[g], med[b]), mad[b]);
    z_arr[g] = z;
    nv += z == z ? 1 : 0;
  }
  nv = warp_sum(nv);
  if (lane == 0 && nv) atomicAdd(&s_nvalid, nv);
  __syncthreads();
  // C6: cutoff = k-th largest non-NaN z (an exact selection by warp 0)
  const int nvalid = s_nvalid;
  const int ksel = min(n_top, nvalid);
  if (warp == 0 && ksel > 0) {
    auto key_z = [&](int i, unsigned long long& key) -> bool {
      const double z = z_arr[i];
      key = dkey(z);
      return z == z;
    };
    const double cut = dkey_inv(warp_select(G, nvalid - ksel + 1, hist[0], key_z));
    if (lane == 0) s_cut = cut;
  }
  __syncthreads();
  const double cut = s_cut;
  for (int g = tid; g < G; g += kHv2Threads) {
    const double z = z_arr[g];
    out_mask[g] = (ksel > 0 && z == z && z >= cut) ? 1 : 0;
  }
  __syncthreads();
  cta_compact(G, out_mask, out_idx, out_count, scan);
}

// ------------------------------------------------------------------ per-batch merge
__global__ void __launch_bounds__(kHv2Threads)
hvg_merge_batches_kernel(int G, int B, const uint8_t* __restrict__ masks, const double* __restrict__ z,
                         int n_top, int32_t* __restrict__ nbat, double* __restrict__ zbar,
                         uint8_t* __restrict__ out_mask, int32_t* __restrict__ out_idx,
                         int32_t* __restrict__ out_count) {
  __shared__ int hist[256];
  __shared__ int lvl[257];                                  // genes per nbatches level
  __shared__ int scan[kHv2Threads + 1];
  __shared__ int s_level, s_tail, s_nn;
  __shared__ double s_cut;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const double kNaN = __longlong_as_double(0x7ff8000000000000ll);
  for (int i = tid; i < 257; i += kHv2Threads) lvl[i] = 0;
  if (tid == 0) { s_nn = 0; s_tail = 0; s_level = 0; s_cut = 0.0; }
  __syncthreads();
  // B1 / B2: batches in the order 0 .. B-1 (a fixed summation order, as the oracle)
  for (int g = tid; g < G; g += kHv2Threads) {
    int nbg = 0, cnt = 0;
    double s = 0.0;
    for (int b = 0; b < B; ++b) {
      nbg += masks[(size_t)b * G + g] ? 1 : 0;
      const double v = z[(size_t)b * G + g];
      if (v == v) { s = __dadd_rn(s, v); ++cnt; }
    }
    nbat[g] = nbg;
    zbar[g] = cnt ? __ddiv_rn(s, (double)cnt) : kNaN;
    atomicAdd(&lvl[nbg], 1);
  }
  __syncthreads();
  // B3: the level that holds the n_top-th gene, then the rank inside it (NaN zbar last)
  const int k = min(n_top, G);
  if (tid == 0 && k > 0) {
    int above = 0, L = B;
    while (L > 0 && above + lvl[L] < k) { above += lvl[L]; --L; }
    s_level = L;
    s_tail = k - above;                                     // rank inside the level, 1-based from the top
  }
  __syncthreads();
  const int L = s_level, r = s_tail;
  if (k > 0) {
    int nn = 0;
    for (int g = tid; g < G; g += kHv2Threads) nn += (nbat[g] == L && zbar[g] == zbar[g]) ? 1 : 0;
    nn = warp_sum(nn);
    if (lane == 0 && nn) atomicAdd(&s_nn, nn);
  }
  __syncthreads();
  const int nn = s_nn;
  const bool in_tail = k > 0 && r > nn;                     // the cutoff sits among the level's NaN genes
  if (warp == 0 && k > 0 && !in_tail) {
    auto key_z = [&](int i, unsigned long long& key) -> bool {
      const double v = zbar[i];
      key = dkey(v);
      return nbat[i] == L && v == v;
    };
    const double cut = dkey_inv(warp_select(G, nn - r + 1, hist, key_z));
    if (lane == 0) s_cut = cut;
  }
  __syncthreads();
  const double cut = s_cut;
  for (int g = tid; g < G; g += kHv2Threads) {
    const int nbg = nbat[g];
    const double v = zbar[g];
    bool sel = false;
    if (k > 0) sel = nbg > L || (nbg == L && (in_tail || (v == v && v >= cut)));
    out_mask[g] = sel ? 1 : 0;
  }
  __syncthreads();
  cta_compact(G, out_mask, out_idx, out_count, scan);
}

// ------------------------------------------------------------------ host side
size_t hvg_cell_ranger_workspace_bytes(int32_t G) {
  const size_t g = (size_t)(G > 0 ? G : 0);
  return 2 * align_up(sizeof(double) * g, 256) + align_up(sizeof(int32_t) * g, 256);
}

int launch_hvg_cell_ranger(int32_t G, const double* mean, const double* var, int32_t n_top, double* out_disp,
                           double* out_disp_norm, int32_t* out_bin, uint8_t* out_mask, int32_t* out_idx,
                           int32_t* out_count, void* ws, cudaStream_t st) {
  unsigned char* w = static_cast<unsigned char*>(ws);
  const size_t gsz = align_up(sizeof(double) * (size_t)G, 256);
  double* d = out_disp ? out_disp : reinterpret_cast<double*>(w);
  double* z = out_disp_norm ? out_disp_norm : reinterpret_cast<double*>(w + gsz);
  int32_t* bin = out_bin ? out_bin : reinterpret_cast<int32_t*>(w + 2 * gsz);
  hvg_cell_ranger_kernel<<<1, kHv2Threads, 0, st>>>(G, mean, var, n_top, d, z, bin, out_mask, out_idx, out_count);
  RSC_LAUNCH_CHECK("hvg_cell_ranger_kernel");
  return RSC_OK;
}

int launch_hvg_merge_batches(int32_t G, int32_t B, const uint8_t* masks, const double* disp_norm, int32_t n_top,
                             int32_t* out_nbatches, double* out_mean, uint8_t* out_mask, int32_t* out_idx,
                             int32_t* out_count, cudaStream_t st) {
  hvg_merge_batches_kernel<<<1, kHv2Threads, 0, st>>>(G, B, masks, disp_norm, n_top, out_nbatches, out_mean, out_mask,
                                                      out_idx, out_count);
  RSC_LAUNCH_CHECK("hvg_merge_batches_kernel");
  return RSC_OK;
}

}  // namespace rsc
