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

constexpr int kHvgBatch = 8;        // elements a thread loads before it uses them (hides L2 latency)
constexpr size_t kHvgPartBytes = 176 * 1024;   // shared memory for the per-bin partial sums
constexpr int kHvgValueBins = 2048; // top-k: equal-width value bins of the first selection pass
constexpr int kHvgMaxCand = 2048;   // top-k: keys of the bin that holds the cutoff
constexpr int kHvgFastRounds = 64;  // compaction: one selection bit per round of 1024 genes

// per-bin statistics: a bin's partial sums live in `slots` thread-private columns of shared
// memory (slots = the largest power of two <= 1024 that fits); 0 = too many bins, warp-per-bin
__host__ __device__ inline int hvg_slots(int n_bins) {
  int slots = kHvgThreads;
  while (slots >= 32 && (size_t)slots * n_bins * sizeof(double) > kHvgPartBytes) slots >>= 1;
  return slots >= 32 ? slots : 0;
}

// shared-memory carve-up (host and device must agree)
struct HvgSmem {
  size_t edges, mu_b, sd_b, red, part_s, part_c, hist, cand, wsum, rcnt, total;
};
__host__ __device__ inline HvgSmem hvg_smem(int G, int n_bins) {
  HvgSmem m;
  size_t o = 0;
  m.edges = o;  o += sizeof(double) * (size_t)(n_bins + 1);
  m.mu_b = o;   o += sizeof(double) * (size_t)n_bins;
  m.sd_b = o;   o += sizeof(double) * (size_t)n_bins;
  m.red = o;    o += sizeof(double) * 2 * kHvgWarps;
  const int slots = hvg_slots(n_bins);                  // 0: warp-per-bin path
  m.part_s = o; o += sizeof(double) * (size_t)slots * n_bins;
  m.part_c = o; o += sizeof(int) * (size_t)(slots ? n_bins : 0);
  o = (o + 7) & ~(size_t)7;
  m.cand = o;   o += sizeof(unsigned long long) * kHvgMaxCand;
  m.hist = o;   o += sizeof(int) * kHvgValueBins;
  m.wsum = o;   o += sizeof(int) * kHvgWarps;
  const int rounds = (G + kHvgThreads - 1) / kHvgThreads;
  m.rcnt = o;   o += sizeof(int) * (size_t)(rounds <= kHvgFastRounds ? rounds * kHvgWarps : 0);
  m.total = (o + 15) & ~(size_t)15;
  return m;
}

// H1 / H2 on many CTAs (two fp64 logarithms per gene are the one compute-heavy part): dispersion
// and transforms of one gene per thread, min / max of the transformed mean per block
constexpr int kHvgTBlock = 256;
__global__ void __launch_bounds__(kHvgTBlock)
hvg_transform_kernel(int G, const double* __restrict__ mean, const double* __restrict__ var, int flags,
                     double* __restrict__ m_arr, double* __restrict__ d_arr, double* __restrict__ blk_mm) {
  __shared__ double s_lo[kHvgTBlock / 32], s_hi[kHvgTBlock / 32];
  const int g = blockIdx.x * kHvgTBlock + threadIdx.x;
  const double kNaN = __longlong_as_double(0x7ff8000000000000ll);
  double lo = __longlong_as_double(0x7ff0000000000000ll), hi = -lo;
  if (g < G) {
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
    lo = m; hi = m;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if ((threadIdx.x & 31) == 0) { s_lo[threadIdx.x >> 5] = lo; s_hi[threadIdx.x >> 5] = hi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < kHvgTBlock / 32; ++w) { lo = fmin(lo, s_lo[w]); hi = fmax(hi, s_hi[w]); }
    blk_mm[2 * blockIdx.x] = lo;
    blk_mm[2 * blockIdx.x + 1] = hi;
  }
}

__global__ void __launch_bounds__(kHvgThreads)
hvg_kernel(int G, const double* __restrict__ blk_mm, int n_tblocks, int n_top,
           int n_bins, int flags, double* __restrict__ m_arr, double* __restrict__ d_arr,
           double* __restrict__ z_arr, int32_t* __restrict__ bin_arr,
           uint8_t* __restrict__ out_mask, int32_t* __restrict__ out_idx,
           int32_t* __restrict__ out_count) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const HvgSmem L = hvg_smem(G, n_bins);
  double* edges = reinterpret_cast<double*>(smem_raw + L.edges);   // n_bins + 1
  double* mu_b = reinterpret_cast<double*>(smem_raw + L.mu_b);     // n_bins
  double* sd_b = reinterpret_cast<double*>(smem_raw + L.sd_b);     // n_bins
  double* red = reinterpret_cast<double*>(smem_raw + L.red);       // 2 * kHvgWarps
  double* part_s = reinterpret_cast<double*>(smem_raw + L.part_s); // n_bins x slots (fast path)
  int* part_c = reinterpret_cast<int*>(smem_raw + L.part_c);       // n_bins: valid genes per bin
  int* hist = reinterpret_cast<int*>(smem_raw + L.hist);           // kHvgValueBins (radix: 256 used)
  unsigned long long* cand = reinterpret_cast<unsigned long long*>(smem_raw + L.cand);   // kHvgMaxCand
  int* wsum = reinterpret_cast<int*>(smem_raw + L.wsum);           // kHvgWarps
  int* rcnt = reinterpret_cast<int*>(smem_raw + L.rcnt);           // rounds x kHvgWarps (fast path)
  __shared__ unsigned long long s_prefix;
  __shared__ int s_remaining, s_nvalid, s_base, s_nonfinite, s_ncand, s_bin;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const double kNaN = __longlong_as_double(0x7ff8000000000000ll);
  constexpr int kStride = kHvgBatch * kHvgThreads;

  // H1 / H2 were done by hvg_transform_kernel; min / max of the transformed mean over its blocks
  double lo = __longlong_as_double(0x7ff0000000000000ll), hi = -lo;
  for (int i = tid; i < n_tblocks; i += kHvgThreads) {
    lo = fmin(lo, blk_mm[2 * i]);
    hi = fmax(hi, blk_mm[2 * i + 1]);
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
  for (int g0 = tid; g0 < G; g0 += kStride) {
    double m8[kHvgBatch];
#pragma unroll
    for (int u = 0; u < kHvgBatch; ++u) {
      const int g = g0 + u * kHvgThreads;
      m8[u] = g < G ? m_arr[g] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < kHvgBatch; ++u) {
      const int g = g0 + u * kHvgThreads;
      int a = 0, b = n_bins - 1;
      while (a < b) {
        const int mid = (a + b) >> 1;
        if (m8[u] <= edges[mid + 1]) b = mid; else a = mid + 1;
      }
      if (g < G) bin_arr[g] = a;
    }
  }
  __syncthreads();

  // H5: per-bin mean and sample sd of the non-NaN dispersions (two passes)
  const int slots = hvg_slots(n_bins);
  if (slots) {
    // every thread adds its genes' values into its OWN column of the bin's row of partial sums
    // (plain read-modify-write, no atomics, no shuffles; threads that share a column take
    // turns, `phases` of them); then one warp per bin adds the row up: a fixed summation order
    const int phases = kHvgThreads / slots;
    const int col = tid & (slots - 1), my_phase = tid / slots;
    for (int pass = 0; pass < 2; ++pass) {
      for (int i = tid; i < slots * n_bins; i += kHvgThreads) part_s[i] = 0.0;
      if (pass == 0) for (int i = tid; i < n_bins; i += kHvgThreads) part_c[i] = 0;
      __syncthreads();
      for (int ph = 0; ph < phases; ++ph) {
        if (ph == my_phase) {
          for (int g0 = tid; g0 - tid < G; g0 += kStride) {   // warp-uniform trip count
            double d8[kHvgBatch];
            int b8[kHvgBatch];
#pragma unroll
            for (int u = 0; u < kHvgBatch; ++u) {
              const int g = g0 + u * kHvgThreads;
              b8[u] = g < G ? bin_arr[g] : 0;
              d8[u] = g < G ? d_arr[g] : kNaN;
            }
#pragma unroll
            for (int u = 0; u < kHvgBatch; ++u) {
              const bool ok = d8[u] == d8[u];             // NaN dispersions are skipped
              if (pass == 0) {                            // genes per bin, one atomic per warp and bin
                const unsigned act = __ballot_sync(0xffffffffu, ok);
                if (ok) {
                  const unsigned same = __match_any_sync(act, b8[u]);
                  if (lane == __ffs(same) - 1) atomicAdd(&part_c[b8[u]], __popc(same));
                }
              }
              if (ok) {
                double v = d8[u];
                if (pass == 1) { const double t = v - mu_b[b8[u]]; v = t * t; }
                part_s[b8[u] * slots + col] += v;
              }
            }
          }
        }
        if (phases > 1) __syncthreads();
      }
      __syncthreads();
      for (int b = warp; b < n_bins; b += kHvgWarps) {
        double sacc = 0.0;
        for (int i = lane; i < slots; i += 32) sacc += part_s[b * slots + i];
        sacc = warp_sum(sacc);
        if (lane == 0) {
          const int c = part_c[b];
          if (pass == 0) {
            mu_b[b] = c ? sacc / (double)c : kNaN;       // the bin's mean (used by pass 1)
          } else {
            const double mk = mu_b[b];
            if (c == 0) { mu_b[b] = kNaN; sd_b[b] = kNaN; }
            else if (c == 1) { mu_b[b] = 0.0; sd_b[b] = mk; }
            else sd_b[b] = sqrt(sacc / (double)(c - 1));
          }
        }
      }
      __syncthreads();
    }
  } else {
    // many bins: one warp per bin, two scans of the genes
    for (int b = warp; b < n_bins; b += kHvgWarps) {
      double sacc = 0.0;
      int c = 0;
      for (int g = lane; g < G; g += 32) {
        if (bin_arr[g] == b) {
          const double d = d_arr[g];
          if (d == d) { sacc += d; ++c; }
        }
      }
      sacc = warp_sum(sacc);
      c = warp_sum(c);
      const double mk = sacc / (double)c;
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
    __syncthreads();
  }
  if (tid == 0) { s_prefix = 0ull; s_nvalid = 0; }
  __syncthreads();

  // H6: z-score; count the valid (non-NaN) genes; range of the finite z
  int nv = 0, nonfin = 0;
  double zlo = __longlong_as_double(0x7ff0000000000000ll), zhi = -zlo;
  if (tid == 0) s_nonfinite = 0;
  for (int g0 = tid; g0 < G; g0 += kStride) {
    double d8[kHvgBatch];
    int b8[kHvgBatch];
#pragma unroll
    for (int u = 0; u < kHvgBatch; ++u) {
      const int g = g0 + u * kHvgThreads;
      b8[u] = g < G ? bin_arr[g] : 0;
      d8[u] = g < G ? d_arr[g] : kNaN;
    }
#pragma unroll
    for (int u = 0; u < kHvgBatch; ++u) {
      const int g = g0 + u * kHvgThreads;
      const double z = __ddiv_rn(__dsub_rn(d8[u], mu_b[b8[u]]), sd_b[b8[u]]);
      if (g < G) {
        z_arr[g] = z;
        if (z == z) {
          ++nv;
          if (isinf(z)) ++nonfin; else { zlo = fmin(zlo, z); zhi = fmax(zhi, z); }
        }
      }
    }
  }
  nv = warp_sum(nv);
  nonfin = warp_sum(nonfin);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    zlo = fmin(zlo, __shfl_xor_sync(0xffffffffu, zlo, o));
    zhi = fmax(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
  }
  __syncthreads();                                        // red[] and s_nonfinite are free / set
  if (lane == 0) {
    if (nv) atomicAdd(&s_nvalid, nv);
    if (nonfin) atomicAdd(&s_nonfinite, nonfin);
    red[warp] = zlo; red[kHvgWarps + warp] = zhi;
  }
  __syncthreads();
  zlo = red[0]; zhi = red[kHvgWarps];
  for (int w = 1; w < kHvgWarps; ++w) { zlo = fmin(zlo, red[w]); zhi = fmax(zhi, red[kHvgWarps + w]); }
  const int k_sel = min(n_top, s_nvalid);

  // H7: exact k-th largest non-NaN z.  Fast path: ONE histogram pass over kHvgValueBins
  // equal-width bins of [zlo, zhi] (z-scores spread over many bins, so the shared atomics do
  // not pile up on a few counters the way the leading radix digits do), the bin holding the
  // cutoff is gathered, and the exact key is found among its few members by rank counting.
  bool selected = k_sel <= 0;
  if (k_sel > 0 && s_nonfinite == 0 && zhi > zlo) {
    const double scale = __ddiv_rn((double)kHvgValueBins - 0.001, __dsub_rn(zhi, zlo));
    auto vbin = [&](double z) -> int {                    // monotone in z
      const int b = (int)__dmul_rn(__dsub_rn(z, zlo), scale);
      return min(max(b, 0), kHvgValueBins - 1);
    };
    for (int i = tid; i < kHvgValueBins; i += kHvgThreads) hist[i] = 0;
    if (tid == 0) s_ncand = 0;
    __syncthreads();
    for (int g0 = tid; g0 < G; g0 += kStride) {
      double z8[kHvgBatch];
#pragma unroll
      for (int u = 0; u < kHvgBatch; ++u) {
        const int g = g0 + u * kHvgThreads;
        z8[u] = g < G ? z_arr[g] : kNaN;
      }
#pragma unroll
      for (int u = 0; u < kHvgBatch; ++u)
        if (z8[u] == z8[u]) atomicAdd(&hist[vbin(z8[u])], 1);
    }
    __syncthreads();
    if (warp == 0) {                                      // bin of the k_sel-th largest; rank inside it
      constexpr int per = kHvgValueBins / 32;
      int tot = 0;
      for (int i = 0; i < per; ++i) tot += hist[lane * per + i];
      int above = 0;                                      // values in the bins of higher lanes
      // plain suffix sum over 32 lanes (tiny): lane l needs sum of tot over lanes > l
      for (int l = 31; l > 0; --l) {
        const int t = __shfl_sync(0xffffffffu, tot, l);
        if (lane < l) above += t;
      }
      if (above < k_sel && k_sel <= above + tot) {        // exactly one lane
        int acc = above;
        for (int i = per - 1; i >= 0; --i) {
          const int c = hist[lane * per + i];
          if (acc + c >= k_sel) { s_bin = lane * per + i; s_remaining = k_sel - acc; break; }
          acc += c;
        }
      }
    }
    __syncthreads();
    const int cbin = s_bin;
    for (int g0 = tid; g0 < G; g0 += kStride) {
      double z8[kHvgBatch];
#pragma unroll
      for (int u = 0; u < kHvgBatch; ++u) {
        const int g = g0 + u * kHvgThreads;
        z8[u] = g < G ? z_arr[g] : kNaN;
      }
#pragma unroll
      for (int u = 0; u < kHvgBatch; ++u) {
        if (z8[u] == z8[u] && vbin(z8[u]) == cbin) {
          const int pos = atomicAdd(&s_ncand, 1);
          if (pos < kHvgMaxCand) cand[pos] = z_key(z8[u]);
        }
      }
    }
    __syncthreads();
    const int nc = s_ncand, rem = s_remaining;
    if (nc <= kHvgMaxCand) {
      for (int i = tid; i < nc; i += kHvgThreads) {       // the rem-th largest key of the bin
        const unsigned long long ki = cand[i];
        int gt = 0, ge = 0;
        for (int jx = 0; jx < nc; ++jx) { const unsigned long long kj = cand[jx]; gt += kj > ki; ge += kj >= ki; }
        if (gt < rem && rem <= ge) s_prefix = ki;         // every such i holds the same key
      }
      selected = true;
    }
    __syncthreads();
  }
  // general path: 8 x 8-bit radix select on the order-preserving keys
  if (!selected) {
    if (tid == 0) { s_remaining = k_sel; s_prefix = 0ull; }
    __syncthreads();
    unsigned long long have_mask = 0ull;
    for (int pass = 7; pass >= 0; --pass) {
      const int shift = pass * 8;
      for (int i = tid; i < 256; i += kHvgThreads) hist[i] = 0;
      __syncthreads();
      const unsigned long long prefix = s_prefix;
      for (int g0 = tid; g0 - tid < G; g0 += kStride) {   // warp-uniform trip count
        double z8[kHvgBatch];
#pragma unroll
        for (int u = 0; u < kHvgBatch; ++u) {
          const int g = g0 + u * kHvgThreads;
          z8[u] = g < G ? z_arr[g] : kNaN;
        }
#pragma unroll
        for (int u = 0; u < kHvgBatch; ++u) {
          if (z8[u] == z8[u]) {
            const unsigned long long key = z_key(z8[u]);
            if ((key & have_mask) == prefix) atomicAdd(&hist[(int)((key >> shift) & 255ull)], 1);
          }
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

  // mask + ascending index list
  const int rounds = (G + kHvgThreads - 1) / kHvgThreads;
  if (rounds <= kHvgFastRounds) {
    // one selection bit per round in a register; per (round, warp) counts -> one scan -> scatter
    unsigned long long selbits = 0ull;
    for (int r0 = 0; r0 < rounds; r0 += kHvgBatch) {
      double z8[kHvgBatch];
#pragma unroll
      for (int u = 0; u < kHvgBatch; ++u) {
        const int g = (r0 + u) * kHvgThreads + tid;
        z8[u] = (r0 + u < rounds && g < G) ? z_arr[g] : kNaN;
      }
#pragma unroll
      for (int u = 0; u < kHvgBatch; ++u) {
        const int r = r0 + u;
        if (r < rounds) {                                 // warp-uniform
          const int g = r * kHvgThreads + tid;
          const bool sel = k_sel > 0 && (z8[u] == z8[u]) && (z_key(z8[u]) >= cut);
          if (g < G) out_mask[g] = sel ? 1 : 0;
          if (sel) selbits |= 1ull << r;
          const unsigned bal = __ballot_sync(0xffffffffu, sel);
          if (lane == 0) rcnt[r * kHvgWarps + warp] = __popc(bal);
        }
      }
    }
    __syncthreads();
    if (warp == 0) {                                      // exclusive scan of rcnt in (round, warp) order
      const int per = rounds;                             // n / 32 entries per lane, contiguous
      int tot = 0;
      for (int i = 0; i < per; ++i) tot += rcnt[lane * per + i];
      int incl = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      int run = incl - tot;
      for (int i = 0; i < per; ++i) {
        const int c = rcnt[lane * per + i];
        rcnt[lane * per + i] = run;
        run += c;
      }
      if (lane == 31) { *out_count = incl; }
    }
    __syncthreads();
    if (out_idx != nullptr) {
      for (int r = 0; r < rounds; ++r) {
        const bool sel = (selbits >> r) & 1ull;
        const unsigned bal = __ballot_sync(0xffffffffu, sel);
        if (sel) out_idx[rcnt[r * kHvgWarps + warp] + __popc(bal & ((1u << lane) - 1u))] = r * kHvgThreads + tid;
      }
    }
  } else {
    // very many genes: ordered block compaction, 1024 genes per round
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
}

bool hvg_cluster_ok(int32_t G, int32_t n_bins);
int launch_hvg_cluster(int32_t G, const double* mean, const double* var, int32_t n_top, int32_t n_bins, int flags,
                       double* m_arr, double* d_arr, double* z_arr, int32_t* b_arr, uint8_t* out_mask,
                       int32_t* out_indices, int32_t* out_count, cudaStream_t st);

size_t hvg_workspace_bytes(int32_t G, int32_t /*n_bins*/) {
  // m, d, z (double) + bin (int32), each 256-byte aligned
  const size_t tb = ((size_t)G + kHvgTBlock - 1) / kHvgTBlock;
  return 3 * align_up(sizeof(double) * (size_t)G, 256) + align_up(sizeof(int32_t) * (size_t)G, 256) +
         align_up(sizeof(double) * 2 * tb, 256);
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
  if (hvg_cluster_ok(G, n_bins) && !g_opt.hvg_single_cta)
    return launch_hvg_cluster(G, mean, var, n_top, n_bins, flags, m_arr, d_arr, z_arr, b_arr, out_mask, out_indices,
                              out_count, st);
  const size_t smem = hvg_smem(G, n_bins).total;
  if (smem > 48 * 1024) {
    RSC_CUDA(cudaFuncSetAttribute(hvg_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)smem));
  }
  const int tb = (G + kHvgTBlock - 1) / kHvgTBlock;
  double* blk_mm = reinterpret_cast<double*>(w + 3 * dsz + align_up(sizeof(int32_t) * (size_t)G, 256));
  hvg_transform_kernel<<<tb, kHvgTBlock, 0, st>>>(G, mean, var, flags, m_arr, d_arr, blk_mm);
  RSC_LAUNCH_CHECK("hvg_transform_kernel");
  hvg_kernel<<<1, kHvgThreads, smem, st>>>(G, blk_mm, tb, n_top, n_bins, flags, m_arr, d_arr, z_arr,
                                           b_arr, out_mask, out_indices, out_count);
  RSC_LAUNCH_CHECK("hvg_kernel");
  return RSC_OK;
}

}  // namespace rsc
