// rsc_hvg_select on a thread-block cluster ("gene selection" on the device, L91; steps
// H1..H7 of DESIGN.md section 3).  The one-CTA kernel of hvg.cu walks G <= 36 k genes with 1024
// threads and re-reads its arrays from L2 in every phase: 84 us (+ 5.5 us for the transforms),
// latency-bound.  Here 8 CTAs of one
// cluster (8192 threads) hold the genes IN REGISTERS (<= 8 per thread) through all phases; what
// the phases need from one another crosses the CTAs through distributed shared memory: per-bin
// partial sums (added in CTA order: deterministic), the value histogram of the top-k (every CTA
// reduces one slice), the candidates of the cutoff bin (appended to CTA 0's list with remote
// atomics), the counts of the ordered compaction.  Nine cluster barriers in all; 39 us on 30 k genes
// (cycles on CTA 0: transforms 12 k, bins 5 k, per-bin statistics 16 k, z 15 k, top-k 21 k, compaction 9 k).
// Serves n_bins <= 32 and G <= 65 536; anything else takes the one-CTA kernel.
#include <cooperative_groups.h>
#include <math.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace rsc {

constexpr int kHcCtas = 8;
constexpr int kHcThreads = 1024;
constexpr int kHcWarps = kHcThreads / 32;
constexpr int kHcPer = 8;                    // genes per thread, at most
constexpr int kHcMaxBins = 32;
constexpr int kHcVBins = 2048;               // value bins of the top-k histogram
constexpr int kHcSlice = kHcVBins / kHcCtas; // histogram bins a CTA reduces
constexpr int kHcMaxCand = 2048;
constexpr int kHcCols = 512;                 // thread-private columns of the per-bin partial sums

__device__ __forceinline__ unsigned long long hc_key(double z) {   // order-preserving, -0.0 canonicalised
  z = z + 0.0;
  const unsigned long long b = (unsigned long long)__double_as_longlong(z);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}

struct HcShared {
  double edges[kHcMaxBins + 1];
  double mu_b[kHcMaxBins], sd_b[kHcMaxBins];
  double cta_sum[kHcMaxBins];                // this CTA's per-bin sums, pass 0 / pass 1 (read by the others)
  double cta_ss[kHcMaxBins];
  int cta_cnt[kHcMaxBins];
  double red_lo, red_hi, red_zlo, red_zhi;   // this CTA's extrema (read by the others)
  int red_nv, red_nonfin;
  double wlo[kHcWarps], whi[kHcWarps];
  int wnv[kHcWarps], wnf[kHcWarps];
  int hist[kHcVBins];                        // this CTA's value histogram (fast path) / radix digits
  int slice_tot[kHcSlice];                   // cluster totals of this CTA's slice
  int slice_sum;
  int tot256[256];                           // radix fallback: cluster totals of the 256 digits
  unsigned long long cand[kHcMaxCand];       // CTA 0: candidates of the cutoff bin; all: a local copy
  int ncand;
  int s_bin, s_rem;
  unsigned long long s_cut;
  int s_rem_radix;
  double all_lo, all_hi;                     // cluster-wide values fetched by one thread
  int all_nv, all_nonfin;
  int rcnt[kHcPer][kHcWarps];                // selected genes per (round, warp)
  int cta_sel;
};

__global__ void __cluster_dims__(kHcCtas, 1, 1) __launch_bounds__(kHcThreads, 1)
hvg_cluster_kernel(int G, const double* __restrict__ mean, const double* __restrict__ var, int n_top,
                   int n_bins, int flags, double* __restrict__ m_arr, double* __restrict__ d_arr,
                   double* __restrict__ z_arr, int32_t* __restrict__ bin_arr, uint8_t* __restrict__ out_mask,
                   int32_t* __restrict__ out_idx, int32_t* __restrict__ out_count) {
  __shared__ HcShared s;
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const double kNaN = __longlong_as_double(0x7ff8000000000000ll);
  const double kInf = __longlong_as_double(0x7ff0000000000000ll);
  auto remote = [&](int r) -> HcShared* { return cluster.map_shared_rank(&s, r); };

  // genes of this thread: g = rank * per * 1024 + u * 1024 + tid (ascending in (rank, u, tid))
  const int per = (G + kHcCtas * kHcThreads - 1) / (kHcCtas * kHcThreads);
  const int gbase = rank * per * kHcThreads + tid;
  double m[kHcPer], d[kHcPer], z[kHcPer];
  int bin[kHcPer];
  bool have[kHcPer];

  // ---- H1 / H2: dispersion and Seurat transforms; extrema of the transformed mean
  double lo = kInf, hi = -kInf;
#pragma unroll
  for (int u = 0; u < kHcPer; ++u) {
    const int g = gbase + u * kHcThreads;
    have[u] = u < per && g < G;
    m[u] = 0.0; d[u] = kNaN; z[u] = kNaN; bin[u] = 0;
    if (have[u]) {
      double mu = mean[g];
      if (mu == 0.0) mu = 1e-12;
      double dd = __ddiv_rn(var[g], mu);
      double mm = mu;
      if (flags & RSC_HVG_SEURAT_LOG) {
        if (dd == 0.0) dd = kNaN;
        dd = log(dd);
        mm = log1p(mu);
      }
      m[u] = mm; d[u] = dd;
      m_arr[g] = mm; d_arr[g] = dd;
      lo = fmin(lo, mm); hi = fmax(hi, mm);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if (lane == 0) { s.wlo[warp] = lo; s.whi[warp] = hi; }
  if (tid == 0) { s.ncand = 0; s.s_cut = 0ull; s.s_bin = 0; s.s_rem = 0; }
  __syncthreads();
  if (warp == 0) {                                        // the 32 warps' extrema: one lane each
    lo = s.wlo[lane]; hi = s.whi[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
      hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (lane == 0) { s.red_lo = lo; s.red_hi = hi; }
  }
  cluster.sync();                                                             // (1)
  // distributed shared memory is slow (~20 B / clock / SM, ~250 cycles): lanes 0..7 of warp 0
  // fetch one CTA's values each, in parallel, and the CTA shares the result
  if (warp == 0) {
    lo = kInf; hi = -kInf;
    if (lane < kHcCtas) { const HcShared* q = remote(lane); lo = q->red_lo; hi = q->red_hi; }
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
      lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
      hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (lane == 0) { s.all_lo = lo; s.all_hi = hi; }
  }
  __syncthreads();
  lo = s.all_lo; hi = s.all_hi;

  // ---- H3: edges, separate multiply and add (no FMA contraction) to match numpy.linspace
  const bool degenerate = (lo == hi);
  if (degenerate) {
    lo = __dsub_rn(lo, lo != 0.0 ? __dmul_rn(0.001, fabs(lo)) : 0.001);
    hi = __dadd_rn(hi, hi != 0.0 ? __dmul_rn(0.001, fabs(hi)) : 0.001);
  }
  const double step = __ddiv_rn(__dsub_rn(hi, lo), (double)n_bins);
  if (tid <= n_bins) {
    double e = (tid == n_bins) ? hi : __dadd_rn(__dmul_rn((double)tid, step), lo);
    if (tid == 0 && !degenerate) e = __dsub_rn(e, __dmul_rn(__dsub_rn(hi, lo), 0.001));
    s.edges[tid] = e;
  }
  __syncthreads();

  // ---- H4: bin(m) = smallest k with m <= edge_{k+1}
#pragma unroll
  for (int u = 0; u < kHcPer; ++u) {
    if (have[u]) {
      int a = 0, b = n_bins - 1;
      while (a < b) {
        const int mid = (a + b) >> 1;
        if (m[u] <= s.edges[mid + 1]) b = mid; else a = mid + 1;
      }
      bin[u] = a;
      bin_arr[gbase + u * kHcThreads] = a;
    }
  }

  // ---- H5: per-bin mean and sample sd of the non-NaN dispersions (two passes).  A thread adds
  // its genes into its OWN column of the bin's row of partial sums (plain read-modify-write, no
  // atomics; threads t and t + 512 share a column and take turns), a warp per bin adds the row
  // up, then the 8 CTAs in order: a fixed summation order.
  extern __shared__ __align__(16) double part[];          // [n_bins][kHcCols]
  const int col = tid & (kHcCols - 1);
  for (int pass = 0; pass < 2; ++pass) {
    for (int i = tid * 2; i < n_bins * kHcCols; i += kHcThreads * 2)
      *reinterpret_cast<double2*>(part + i) = make_double2(0.0, 0.0);
    if (pass == 0 && tid < n_bins) s.cta_cnt[tid] = 0;
    __syncthreads();
    for (int ph = 0; ph < kHcThreads / kHcCols; ++ph) {
      if ((tid / kHcCols) == ph) {
#pragma unroll
        for (int u = 0; u < kHcPer; ++u) {
          if (have[u] && d[u] == d[u]) {
            double v = d[u];
            if (pass == 1) { const double t = v - s.mu_b[bin[u]]; v = t * t; }
            part[bin[u] * kHcCols + col] += v;
          }
        }
      }
      __syncthreads();
    }
    if (pass == 0) {                                      // genes per bin: one atomic per warp and bin
#pragma unroll
      for (int u = 0; u < kHcPer; ++u) {
        const bool ok = have[u] && d[u] == d[u];
        const unsigned act = __ballot_sync(0xffffffffu, ok);
        if (ok) {
          const unsigned same = __match_any_sync(act, bin[u]);
          if (lane == __ffs(same) - 1) atomicAdd(&s.cta_cnt[bin[u]], __popc(same));
        }
      }
    }
    for (int b = warp; b < n_bins; b += kHcWarps) {
      double v = 0.0;
      for (int i = lane; i < kHcCols; i += 32) v += part[b * kHcCols + i];
      v = warp_sum(v);
      if (lane == 0) { if (pass == 0) s.cta_sum[b] = v; else s.cta_ss[b] = v; }
    }
    cluster.sync();                                                           // (2), (3)
    if (tid < n_bins) {
      double v = 0.0;
      int c = 0;
      for (int r = 0; r < kHcCtas; ++r) {
        const HcShared* q = remote(r);
        v += pass == 0 ? q->cta_sum[tid] : q->cta_ss[tid];
        c += q->cta_cnt[tid];
      }
      if (pass == 0) {
        s.mu_b[tid] = c ? v / (double)c : kNaN;           // the bin's mean (used by pass 1)
      } else {
        const double mk = s.mu_b[tid];
        if (c == 0) { s.mu_b[tid] = kNaN; s.sd_b[tid] = kNaN; }
        else if (c == 1) { s.mu_b[tid] = 0.0; s.sd_b[tid] = mk; }
        else s.sd_b[tid] = sqrt(v / (double)(c - 1));
      }
    }
    __syncthreads();
  }

  // ---- H6: z-score; valid (non-NaN) genes; range of the finite z
  int nv = 0, nonfin = 0;
  double zlo = kInf, zhi = -kInf;
#pragma unroll
  for (int u = 0; u < kHcPer; ++u) {
    if (have[u]) {
      const double zz = __ddiv_rn(__dsub_rn(d[u], s.mu_b[bin[u]]), s.sd_b[bin[u]]);
      z[u] = zz;
      z_arr[gbase + u * kHcThreads] = zz;
      if (zz == zz) {
        ++nv;
        if (isinf(zz)) ++nonfin; else { zlo = fmin(zlo, zz); zhi = fmax(zhi, zz); }
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
  if (lane == 0) { s.wlo[warp] = zlo; s.whi[warp] = zhi; s.wnv[warp] = nv; s.wnf[warp] = nonfin; }
  for (int i = tid; i < kHcVBins; i += kHcThreads) s.hist[i] = 0;
  __syncthreads();
  if (warp == 0) {
    zlo = s.wlo[lane]; zhi = s.whi[lane];
    int a = s.wnv[lane], b = s.wnf[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      zlo = fmin(zlo, __shfl_xor_sync(0xffffffffu, zlo, o));
      zhi = fmax(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
      a += __shfl_xor_sync(0xffffffffu, a, o);
      b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    if (lane == 0) { s.red_zlo = zlo; s.red_zhi = zhi; s.red_nv = a; s.red_nonfin = b; }
  }
  cluster.sync();                                                             // (4)
  if (warp == 0) {
    int a = 0, b = 0;
    zlo = kInf; zhi = -kInf;
    if (lane < kHcCtas) {
      const HcShared* q = remote(lane);
      zlo = q->red_zlo; zhi = q->red_zhi; a = q->red_nv; b = q->red_nonfin;
    }
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
      zlo = fmin(zlo, __shfl_xor_sync(0xffffffffu, zlo, o));
      zhi = fmax(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
      a += __shfl_xor_sync(0xffffffffu, a, o);
      b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    if (lane == 0) { s.all_lo = zlo; s.all_hi = zhi; s.all_nv = a; s.all_nonfin = b; }
  }
  __syncthreads();
  zlo = s.all_lo; zhi = s.all_hi;
  const int nvalid = s.all_nv, n_nonfin = s.all_nonfin;
  const int k_sel = min(n_top, nvalid);

  // ---- H7: exact k-th largest non-NaN z
  bool selected = k_sel <= 0;
  if (k_sel > 0 && n_nonfin == 0 && zhi > zlo) {
    // fast path: ONE histogram over kHcVBins equal-width bins of [zlo, zhi]; every CTA reduces a
    // slice of it, the bin holding the cutoff is found from the slice sums, its members are
    // gathered in CTA 0 and the exact key is found among them by rank counting
    const double scale = __ddiv_rn((double)kHcVBins - 0.001, __dsub_rn(zhi, zlo));
    auto vbin = [&](double zz) -> int {                   // monotone in z
      const int b = (int)__dmul_rn(__dsub_rn(zz, zlo), scale);
      return min(max(b, 0), kHcVBins - 1);
    };
#pragma unroll
    for (int u = 0; u < kHcPer; ++u)
      if (have[u] && z[u] == z[u]) atomicAdd(&s.hist[vbin(z[u])], 1);
    cluster.sync();                                                           // (5) all local histograms complete
    if (tid < kHcSlice) {
      int t = 0;
      for (int r = 0; r < kHcCtas; ++r) t += remote(r)->hist[rank * kHcSlice + tid];
      s.slice_tot[tid] = t;
    }
    __syncthreads();
    if (warp == 0) {
      int t = 0;
      for (int i = lane; i < kHcSlice; i += 32) t += s.slice_tot[i];
      t = warp_sum(t);
      if (lane == 0) s.slice_sum = t;
    }
    cluster.sync();                                                           // (6) slice totals complete
    if (warp == 0) {
      // the slice (from the top) that holds the k_sel-th largest, then the bin inside it
      const int mysum = lane < kHcCtas ? remote(lane)->slice_sum : 0;
      int above = 0, rs = kHcCtas - 1;
      for (; rs > 0; --rs) {
        const int t = __shfl_sync(0xffffffffu, mysum, rs);
        if (above + t >= k_sel) break;
        above += t;
      }
      const HcShared* q = remote(rs);
      constexpr int pl = kHcSlice / 32;                   // bins per lane
      int c[pl], tot = 0;
#pragma unroll
      for (int i = 0; i < pl; ++i) { c[i] = q->slice_tot[lane * pl + i]; tot += c[i]; }
      int hi_lanes = 0;                                   // values in the bins of higher lanes
      for (int l = 31; l > 0; --l) {
        const int t = __shfl_sync(0xffffffffu, tot, l);
        if (lane < l) hi_lanes += t;
      }
      const int ab = above + hi_lanes;
      if (ab < k_sel && k_sel <= ab + tot) {              // exactly one lane
        int acc = ab;
#pragma unroll
        for (int i = pl - 1; i >= 0; --i) {
          if (acc >= 0 && acc + c[i] >= k_sel) { s.s_bin = rs * kHcSlice + lane * pl + i; s.s_rem = k_sel - acc; acc = -0x40000000; }
          else if (acc >= 0) acc += c[i];
        }
      }
    }
    __syncthreads();
    const int cbin = s.s_bin;
    HcShared* q0 = remote(0);
#pragma unroll
    for (int u = 0; u < kHcPer; ++u) {
      if (have[u] && z[u] == z[u] && vbin(z[u]) == cbin) {
        const int pos = atomicAdd(&q0->ncand, 1);         // remote shared-memory atomic
        if (pos < kHcMaxCand) q0->cand[pos] = hc_key(z[u]);
      }
    }
    cluster.sync();                                                           // (7) candidate list complete
    if (tid == 0) s.all_nv = q0->ncand;
    __syncthreads();
    const int nc = s.all_nv, rem = s.s_rem;
    if (nc <= kHcMaxCand) {
      if (rank != 0)
        for (int i = tid; i < nc; i += kHcThreads) s.cand[i] = q0->cand[i];   // local copy
      __syncthreads();
      for (int i = tid; i < nc; i += kHcThreads) {        // the rem-th largest key of the bin
        const unsigned long long ki = s.cand[i];
        int gt = 0, ge = 0;
        for (int jx = 0; jx < nc; ++jx) { const unsigned long long kj = s.cand[jx]; gt += kj > ki; ge += kj >= ki; }
        if (gt < rem && rem <= ge) s.s_cut = ki;          // every such i holds the same key
      }
      selected = true;
    }
    __syncthreads();
  }
  if (!selected) {
    // general path (non-finite z, a constant z, or too many ties in one bin): 8 x 8-bit radix
    // select on the order-preserving keys, the digit histogram summed over the cluster
    unsigned long long prefix = 0ull, have_mask = 0ull;
    int rem = k_sel;
    for (int pass = 7; pass >= 0; --pass) {
      const int shift = pass * 8;
      for (int i = tid; i < 256; i += kHcThreads) s.hist[i] = 0;
      __syncthreads();
#pragma unroll
      for (int u = 0; u < kHcPer; ++u) {
        if (have[u] && z[u] == z[u]) {
          const unsigned long long key = hc_key(z[u]);
          if ((key & have_mask) == prefix) atomicAdd(&s.hist[(int)((key >> shift) & 255ull)], 1);
        }
      }
      cluster.sync();
      if (tid < 256) {
        int t = 0;
        for (int r = 0; r < kHcCtas; ++r) t += remote(r)->hist[tid];
        s.tot256[tid] = t;
      }
      __syncthreads();
      if (tid == 0) {
        int rr = rem, dgt = 255;
        for (; dgt > 0; --dgt) {
          if (s.tot256[dgt] >= rr) break;
          rr -= s.tot256[dgt];
        }
        s.s_rem_radix = rr;
        s.s_cut = prefix | ((unsigned long long)dgt << shift);
      }
      __syncthreads();
      rem = s.s_rem_radix;
      prefix = s.s_cut;
      have_mask |= (255ull << shift);
      cluster.sync();                                     // the digit histograms may be cleared again
    }
  }
  const unsigned long long cut = s.s_cut;

  // ---- mask + ascending index list: per (round, warp) counts, one scan per CTA, CTA offsets
  // from the cluster
  unsigned selbits = 0u;
#pragma unroll
  for (int u = 0; u < kHcPer; ++u) {
    const bool sel = have[u] && k_sel > 0 && (z[u] == z[u]) && (hc_key(z[u]) >= cut);
    if (have[u]) out_mask[gbase + u * kHcThreads] = sel ? 1 : 0;
    if (sel) selbits |= 1u << u;
    const unsigned bal = __ballot_sync(0xffffffffu, sel);
    if (lane == 0) s.rcnt[u][warp] = __popc(bal);
  }
  __syncthreads();
  if (warp == 0) {                                        // exclusive scan of rcnt in (round, warp) order
    constexpr int pl = kHcPer * kHcWarps / 32;            // 8 entries per lane, contiguous
    int* rc = &s.rcnt[0][0];
    int tot = 0;
#pragma unroll
    for (int i = 0; i < pl; ++i) tot += rc[lane * pl + i];
    int incl = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    int run = incl - tot;
#pragma unroll
    for (int i = 0; i < pl; ++i) {
      const int c = rc[lane * pl + i];
      rc[lane * pl + i] = run;
      run += c;
    }
    if (lane == 31) s.cta_sel = incl;
  }
  cluster.sync();                                                             // (8) CTA totals complete
  if (warp == 0) {
    const int t = lane < kHcCtas ? remote(lane)->cta_sel : 0;
    int o = lane < rank ? t : 0, total = t;
#pragma unroll
    for (int k = 4; k > 0; k >>= 1) {
      o += __shfl_xor_sync(0xffffffffu, o, k);
      total += __shfl_xor_sync(0xffffffffu, total, k);
    }
    if (lane == 0) { s.all_nv = o; if (rank == 0) *out_count = total; }
  }
  __syncthreads();
  const int off = s.all_nv;
  if (out_idx != nullptr) {
#pragma unroll
    for (int u = 0; u < kHcPer; ++u) {
      const bool sel = (selbits >> u) & 1u;
      const unsigned bal = __ballot_sync(0xffffffffu, sel);
      if (sel) out_idx[off + s.rcnt[u][warp] + __popc(bal & ((1u << lane) - 1u))] = gbase + u * kHcThreads;
    }
  }
  cluster.sync();                                                             // (9) nobody reads a CTA that has exited
}

bool hvg_cluster_ok(int32_t G, int32_t n_bins) {
  return n_bins >= 1 && n_bins <= kHcMaxBins && G >= 1 && G <= kHcCtas * kHcThreads * kHcPer;
}

int launch_hvg_cluster(int32_t G, const double* mean, const double* var, int32_t n_top, int32_t n_bins, int flags,
                       double* m_arr, double* d_arr, double* z_arr, int32_t* b_arr, uint8_t* out_mask,
                       int32_t* out_indices, int32_t* out_count, cudaStream_t st) {
  const size_t dyn = sizeof(double) * (size_t)n_bins * kHcCols;
  RSC_CUDA(cudaFuncSetAttribute(hvg_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
  hvg_cluster_kernel<<<kHcCtas, kHcThreads, dyn, st>>>(G, mean, var, n_top, n_bins, flags, m_arr, d_arr, z_arr, b_arr,
                                                     out_mask, out_indices, out_count);
  RSC_LAUNCH_CHECK("hvg_cluster_kernel");
  return RSC_OK;
}

}  // namespace rsc
