// rsc_normalize_log1p_moments, streaming kernel: x' = x * scale_i, x'' = log1p(x') written
// back, per-gene sums of x'' / x''^2 (log scale) and x' / x'^2 (linear scale) accumulated on
// chip.  PAPER.md:L91 (normalize_total, log1p, "per-gene mean and variance, computed using a
// custom GPU reduction kernel that operates directly on sparse matrices"), L137; the fusion
// itself is BASELINE.json north_star's, not the paper's.  12 B / nnz of DRAM traffic.
//
// Design:
//   * Gene-range groups.  G genes x 20..40 B of accumulators do not fit one SM's shared
//     memory, so the columns are cut into groups of `fine_per_group` blocks of
//     RSC_SPLIT_WIDTH genes; a CTA serves ONE group and keeps that group's accumulators
//     (<= 227 KB) private.  Rows are sorted, so a group's entries are one contiguous
//     segment of every row, located through the row split table (written by the QC pass or
//     by row_splits_kernel).  CTAs are dealt to groups in proportion to the groups' nnz
//     (fused_plan_kernel, on the device), rows to a group's CTAs by an atomic cursor.
//   * Segments are walked in 16-byte aligned quads: one 128-bit load per array and one
//     128-bit store per lane; only the first / last quad of a segment can be partial and
//     takes scalar accesses.
//   * Accumulators: integer sums.  Only 32-bit integer shared atomics are native on
//     sm_100 (ATOMS.ADD; 64-bit and floating-point ones are CAS loops), so a value v is
//     first scaled by a power of two 2^k (chosen on the device) such that a = v * 2^k is an
//     exact integer for every v >= 2^(23-k) -- the float32 significand has 24 bits.
//     LINEAR-scale set (x', a 2^14-fold value range): 5 words per gene,
//         S1 += a      as a 64-bit  integer in two   u32 words (w0, w1)
//         S2 += a * a  as a 96-bit  integer in three u32 words (s0, s1, s2)
//     where a word's carry-out (seen in the value the atomic returns) is added to the next
//     word with a predicated increment: 2^23 <= a < 2^32 takes ~3.1 atomics per entry,
//     2^32 <= a < 2^42 the same path with a two-word a.
//     LOG-scale set (x'' = log1p(x') lies in [log1p(s / T_max), log1p(s)], a few binades):
//     3 words per gene and NO branches -- window 2^23 <= a < 2^28 (32-fold, placed on the
//     device from the cell depths),
//         w0 += a                                  (returning atomic -> carry c1)
//         s0 += low word of b,  b = (a*a + 2^7) >> 8     (returning atomic -> carry c0)
//         W  += high word of b + c0 + (c1 << 26)   (one non-returning atomic)
//     W packs the upper part of S2 (bits 0..25) and the carry count of S1 (bits 26..31); a
//     gene leaves the table when a field is half full (check_tables), so neither can overflow.
//     S1 is exact; S2 is the sum of a*a rounded to a multiple of 2^8, i.e. to <= 2^-39 of the
//     SMALLEST possible a*a (1.8e-12; 1e-13 for a typical x'' of 1..2) -- and still an integer
//     sum.  12 B / gene: 30 k genes need 2 groups, 18 k genes one.
//     Values outside a set's window (or negative / NaN) go to the global double sums directly.
//     Integer adds commute, so the on-chip sums do not depend on the order of the adds; a
//     flush adds every word to its own 64-bit global counter, converted to double once at the
//     end (fused_finish_kernel): bit-reproducible moments.
//   * RSC_MOMENTS_FP64_ACC selects plain double accumulators (CAS atomics) instead: any
//     value range, slower (fused_stream_fp64_kernel).
#include <math.h>

#include <type_traits>

#include "common.cuh"
#include "fused_acc.cuh"

namespace rsc {

// ------------------------------------------------------------------ largest cell total
__global__ void __launch_bounds__(256)
fused_tmax_kernel(FusedPlan* plan, int64_t n_rows, const int64_t* __restrict__ cell_total, float target_sum) {
  __shared__ unsigned int hist[64];
  if (threadIdx.x < 64) hist[threadIdx.x] = 0u;
  __syncthreads();
  long long m = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_rows;
       i += (int64_t)gridDim.x * blockDim.x) {
    const long long t = (long long)cell_total[i];
    m = max(m, t);
    if (t > 0) {
      // the smallest x'' of the cell: a unit count.  Binade of log1p(s / T) (frexp exponent - 1)
      int e;
      frexpf(log1pf(__fdiv_rn(target_sum, (float)t)), &e);
      atomicAdd(&hist[min(max(e - 1 + 32, 0), 63)], 1u);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(&plan->tmax, (unsigned long long)m);
  __syncthreads();
  if (threadIdx.x < 64 && hist[threadIdx.x]) atomicAdd(&plan->depth_hist[threadIdx.x], hist[threadIdx.x]);
}

// floor(log2(x)) for finite x > 0
__device__ __forceinline__ int floor_log2(double x) {
  int e;
  frexp(x, &e);                                            // x = m 2^e, m in [0.5, 1)
  return e - 1;
}

__device__ inline MomentScale make_scale(double v_min, double v_max) {
  // window bottom 2^L <= v_min (so that every expected value converts exactly), but no more
  // than kMaxRangeBits binades below the top 2^E > v_max
  int E;
  frexp(v_max, &E);
  int L = floor_log2(v_min);
  if (L < E - kMaxRangeBits) L = E - kMaxRangeBits;
  if (L > E - 9) L = E - 9;                                // nothing gained by a narrower window
  int k = 23 - L;
  if (k > 100) k = 100;
  if (k < -60) k = -60;
  MomentScale s;
  s.mult = (float)ldexp(1.0, k);
  s.pad = 0.0f;
  s.inv1 = ldexp(1.0, -k);
  s.inv2 = ldexp(1.0, -2 * k);
  return s;
}

// CTAs are dealt to the gene groups in proportion to their cost (one thread).  Cost of a group
// = its entries + a per-row overhead (every CTA of the group walks a segment of EVERY row:
// grab, metadata, edge steps ~ the work of kRowCost entries), so a group of few, sparse columns
// still gets the CTAs its row count needs.
__device__ inline void deal_ctas(FusedPlan* plan, double* mass, int ng, int grid, long long n_rows) {
  double total = 0.0;
  for (int c = 0; c < ng; ++c) { mass[c] += (double)n_rows * kRowCost; total += mass[c]; }
  int n[kMaxGroups];
  int sum = 0;
  for (int c = 0; c < ng; ++c) {
    const double share = total > 0.0 ? mass[c] / total : 1.0 / ng;
    mass[c] = share + 1e-9;
    n[c] = max(1, (int)(share * grid));
    sum += n[c];
  }
  while (sum < grid) {                                   // most loaded group gets the next CTA
    int best = 0;
    for (int c = 1; c < ng; ++c) if (mass[c] / n[c] > mass[best] / n[best]) best = c;
    ++n[best]; ++sum;
  }
  while (sum > grid) {                                   // only if many groups got the floor of 1
    int best = -1;
    for (int c = 0; c < ng; ++c)
      if (n[c] > 1 && (best < 0 || mass[c] / (n[c] - 1) < mass[best] / (n[best] - 1))) best = c;
    --n[best]; --sum;
  }
  plan->n_groups = ng;
  int acc = 0;
  for (int c = 0; c < ng; ++c) { plan->cta_first[c] = acc; acc += n[c]; plan->row_counter[c] = 0ull; }
  plan->cta_first[ng] = acc;
}

// ------------------------------------------------------------------ plan (1 CTA)
__global__ void __launch_bounds__(1024)
fused_plan_kernel(FusedPlan* plan, int G, int K, int fine_per_group, int grid, float target_sum,
                  long long n_rows, const int32_t* __restrict__ gene_n_cells) {
  __shared__ double mass[kMaxGroups];
  const int tid = threadIdx.x;
  const int ng = (K + fine_per_group - 1) / fine_per_group;
  if (tid < kMaxGroups) mass[tid] = 0.0;
  __syncthreads();
  for (int c = 0; c < ng; ++c) {                          // group c = blocks [c K / ng, (c + 1) K / ng)
    const int g0 = ((c * K) / ng) << RSC_SPLIT_SHIFT;
    const int g1 = min(G, (((c + 1) * K) / ng) << RSC_SPLIT_SHIFT);
    double m = 0.0;
    for (int g = g0 + tid; g < g1; g += 1024) {
      const int v = gene_n_cells ? gene_n_cells[g] : 1;
      m += (double)(v > 0 ? v : 0);
    }
    m = warp_sum(m);
    if ((tid & 31) == 0 && m != 0.0) atomicAdd(&mass[c], m);
  }
  __syncthreads();
  if (tid == 0) deal_ctas(plan, mass, ng, grid, n_rows);
  if (tid == 32) {
    // power-of-two scales of the integer accumulators: x' of a unit count in the deepest
    // cell is target_sum / T_max; nothing exceeds target_sum (non-negative data)
    const unsigned long long tm = plan->tmax;
    const double ts = (double)target_sum;
    const float smin_f = tm != 0ull ? __fdiv_rn(target_sum, (float)(long long)tm) : 1.0f;
    double smin = (double)smin_f;
    if (!(smin > 0.0) || !isfinite(smin)) smin = 1.0;
    if (smin > ts) smin = ts;
    plan->sc_lin = make_scale(smin, ts);
    {
      // log-scale set: a window of kLogBinades binades [2^L, 2^(L + kLogBinades)).  The bottom
      // is the binade of the smallest x'' of the data -- a unit count in the deepest cell --
      // taken robustly: the ~n / 65 536 deepest cells are ignored (their small values take the
      // global path), so one outlier cell cannot drag the window away from the bulk.  Never
      // above the top 2^E > log1p(target_sum) (the largest x'' non-negative data can produce),
      // and never below 2^-2: log1p_ge_quarter of an x' < 0.25 is < 0.2232, so such a value
      // fails the window test by itself and the log-only kernel needs no separate x' test.
      int E;
      frexp(log1p(ts) * 1.000001, &E);
      int L = E - kLogBinades;
      {
        // (n / 65 536 cells, at least 8 when the matrix has 4 096 cells or more; was n / 4 096.  Every unit count of
        // an ignored cell takes the per-entry slow path, ~100 us per row segment for one warp: with 24 such rows
        // config 2 had a straggler tail of 25 %; fewer values on the order-dependent global path, too)
        unsigned long long skip = (unsigned long long)n_rows / 65536ull;
        if (skip < 8ull) skip = (unsigned long long)n_rows / 512ull < 8ull ? (unsigned long long)n_rows / 512ull : 8ull;
        unsigned long long below = 0ull;
        for (int b = 0; b < 64; ++b) {
          below += plan->depth_hist[b];
          if (below > skip) { L = min(b - 32, E - kLogBinades); break; }
        }
      }
      L = max(L, -2);
      const int k = 23 - L;
      MomentScale s;
      s.mult = (float)ldexp(1.0, k);
      s.pad = 0.0f;
      s.inv1 = ldexp(1.0, -k);
      s.inv2 = ldexp(1.0, kLogShift - 2 * k);
      plan->sc_log = s;
    }
  }
}

// ------------------------------------------------------------------ plan of the moments-only pass
// rsc_gene_moments knows nothing about the values, so the plan looks at a sample (32 768 stored
// entries in 1 024 clusters spread evenly over the matrix): largest value v_max, smallest positive value, and how
// the entries spread over the column blocks.
//   * 2^E > v_max of the sample;
//   * if at most one sampled value in 1024 lies below 2^(E - kLogBinades), the three-word scheme
//     with the window [2^(E - kLogBinades), 2^E) (12 B / gene), else the five-word scheme (one
//     binade of head room: one-word values 2^(E-8) .. 2^(E+1), two-word values up to 2^(E+11));
//   * gene groups as large as the table allows, CTAs dealt by the sampled entry counts.
// A value the sample did not foresee still lands in the global double sums: correct, only slow.
__global__ void __launch_bounds__(1024)
moments_plan_kernel(FusedPlan* plan, int G, int K, int grid, long long n_rows, long long nnz,
                    const int32_t* __restrict__ indices, const float* __restrict__ data) {
  __shared__ double mass[kMaxGroups];
  __shared__ float s_max[32];
  __shared__ int s_ng, s_E, s_below, s_pos;
  constexpr int kPer = 32;
  const int tid = threadIdx.x;
  // 32 * kPer clusters of 32 consecutive entries (a warp reads one line per load), spread evenly
  const long long step = nnz > 1024LL * kPer ? (nnz - 32) / (32LL * kPer) : 32;
  float vmax = 0.0f;
  int32_t col[kPer];                                      // the sampled entries' columns and values (registers)
  float val[kPer];
#pragma unroll
  for (int i = 0; i < kPer; ++i) {                        // independent loads: all in flight together
    const long long p = ((long long)i * 32 + (tid >> 5)) * step + (tid & 31);
    float v = 0.0f;
    col[i] = -1;
    if (p < nnz) { v = __ldg(data + p); col[i] = __ldg(indices + p); }
    val[i] = v;
    if (v > vmax) vmax = v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
  if ((tid & 31) == 0) s_max[tid >> 5] = vmax;
  if (tid < kMaxGroups) mass[tid] = 0.0;
  if (tid == 0) { s_below = 0; s_pos = 0; }
  __syncthreads();
  if (tid == 0) {
    for (int w = 1; w < 32; ++w) vmax = fmaxf(vmax, s_max[w]);
    if (!(vmax > 0.0f) || !isfinite(vmax)) vmax = 1.0f;
    int E;
    frexp((double)vmax * 1.0000001, &E);                   // 2^E > v_max of the sample
    s_E = E;
  }
  __syncthreads();
  {
    // how much of the sample lies below the narrow window [2^(E - kLogBinades), 2^E)?  Up to one
    // entry in 1024 may (such values take the global double sums: correct, only slower), so a
    // few deep cells do not force the five-word scheme on everybody else
    const float bottom = ldexpf(1.0f, s_E - kLogBinades);
    int below = 0, pos = 0;
#pragma unroll
    for (int i = 0; i < kPer; ++i) {
      pos += val[i] > 0.0f ? 1 : 0;
      below += (val[i] > 0.0f && val[i] < bottom) ? 1 : 0;
    }
    below = warp_sum(below);
    pos = warp_sum(pos);
    if ((tid & 31) == 0) { atomicAdd(&s_below, below); atomicAdd(&s_pos, pos); }
  }
  __syncthreads();
  if (tid == 0) {
    const int E = s_E;
    const bool narrow = (long long)s_below * 1024 <= (long long)s_pos;
    MomentScale sc;
    sc.pad = 0.0f;
    int bpg;
    if (narrow) {
      const int k = 23 - (E - kLogBinades);
      sc.mult = (float)ldexp(1.0, k); sc.inv1 = ldexp(1.0, -k); sc.inv2 = ldexp(1.0, kLogShift - 2 * k);
      plan->sc_log = sc;
      bpg = kLogWords * 4;
    } else {
      const int k = 32 - (E + 1);                          // one binade of head room over the sample
      sc.mult = (float)ldexp(1.0, k); sc.inv1 = ldexp(1.0, -k); sc.inv2 = ldexp(1.0, -2 * k);
      plan->sc_lin = sc;
      bpg = kSetWords * 4;
    }
    plan->scheme = narrow ? 1 : 2;
    const int fit = (int)((kMaxDynSmem - 64) / ((size_t)bpg * RSC_SPLIT_WIDTH));
    const int ng = (K + fit - 1) / fit;
    plan->Gt = ((K + ng - 1) / ng) * RSC_SPLIT_WIDTH;
    plan->n_need = ng + 1;
    for (int c = 0; c <= ng; ++c) plan->need[c] = (c * K) / ng;
    s_ng = ng;
  }
  __syncthreads();
  const int ng = s_ng;
  for (int c = 0; c < ng; ++c) {                          // sampled entries per group
    const int b0 = plan->need[c], b1 = plan->need[c + 1];
    int cnt = 0;
#pragma unroll
    for (int i = 0; i < kPer; ++i) {
      const int b = col[i] >> RSC_SPLIT_SHIFT;
      cnt += (col[i] >= 0 && b >= b0 && b < b1) ? 1 : 0;
    }
    cnt = warp_sum(cnt);
    if ((tid & 31) == 0 && cnt) atomicAdd(&mass[c], (double)cnt);
  }
  __syncthreads();
  if (tid == 0) {
    double tot = 0.0;
    for (int c = 0; c < ng; ++c) tot += mass[c];
    for (int c = 0; c < ng; ++c) mass[c] = tot > 0.0 ? mass[c] / tot * (double)nnz : (double)nnz / ng;
    deal_ctas(plan, mass, ng, grid, n_rows);
  }
}

// Compact row split table of the moments-only pass: out[row][c] = number of the row's entries
// with column < need[c] * RSC_SPLIT_WIDTH, c = 0 .. n_groups.  One thread per row; every interior
// bound is bracketed around the position a uniform spread of the columns predicts (widened
// geometrically), then bisected: a few probes, nearly all in one line.
__global__ void __launch_bounds__(256)
row_splits_compact_kernel(int64_t n_rows, int G, const int64_t* __restrict__ indptr,
                          const int32_t* __restrict__ indices, const FusedPlan* __restrict__ plan,
                          uint32_t* __restrict__ out) {
  const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (row >= n_rows) return;
  const int ng = plan->n_groups;
  const int64_t beg = indptr[row];
  const int len = (int)(indptr[row + 1] - beg);
  uint32_t* o = out + (size_t)row * kNeedStride;
  o[0] = 0u;
  for (int c = 1; c < ng; ++c) {
    const int32_t bound = plan->need[c] << RSC_SPLIT_SHIFT;
    int w = 16;
    const int guess = (int)(((long long)len * bound) / G);
    int lo = max(guess - w, 0), hi = min(guess + w, len);
    while (lo > 0 && __ldg(indices + beg + lo - 1) >= bound) { hi = lo - 1; w *= 2; lo = max(lo - w, 0); }
    while (hi < len && __ldg(indices + beg + hi) < bound) { lo = hi + 1; w *= 2; hi = min(hi + w, len); }
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (__ldg(indices + beg + mid) < bound) lo = mid + 1; else hi = mid;
    }
    o[c] = (uint32_t)lo;
  }
  o[ng] = (uint32_t)len;
}

// ------------------------------------------------------------------ streaming kernel
// MOM = false: the fused pass (x' = x * scale_i, x'' = log1p(x') written back, sums of x'' / x').
// MOM = true: the moments-only pass of rsc_gene_moments (transform 0): the value is x itself,
// nothing is written back, exactly one set is active (LOG = the three-word scheme, LIN = the
// five-word scheme), the gene groups and the table size come from the plan (device memory),
// and the split table is the compact one ([kNeedStride] entries per row).
template <bool LOG, bool LIN, bool MOM>
__device__ __forceinline__ void fused_stream_body(const FusedArgs& a, uint32_t* fsm, unsigned& s_rows) {
  const int tid = threadIdx.x, lane = tid & 31;
  const int Gt = MOM ? a.plan->Gt : a.Gt;
  const int K = a.n_fine;

  // which group does this CTA serve?
  const FusedPlan* plan = a.plan;
  int grp = 0;
  {
    const int ng = plan->n_groups;
    while (grp + 1 < ng && (int)blockIdx.x >= plan->cta_first[grp + 1]) ++grp;
  }
  const float mult_log = plan->sc_log.mult, mult_lin = plan->sc_lin.mult;
  // group = blocks [grp K / ng, (grp + 1) K / ng) (fused) or [need[grp], need[grp + 1]) (moments-only)
  const int f0 = MOM ? plan->need[grp] : (grp * K) / plan->n_groups;
  const int f1 = MOM ? plan->need[grp + 1] : ((grp + 1) * K) / plan->n_groups;
  const int s0i = MOM ? grp : f0, s1i = MOM ? grp + 1 : f1;     // the row's split entries to read
  const size_t sstride = MOM ? (size_t)kNeedStride : (size_t)(K + 1);
  const int g0 = f0 << RSC_SPLIT_SHIFT;
  const int ng_genes = min(a.n_cols, f1 << RSC_SPLIT_SHIFT) - g0;
  unsigned long long* counter = &a.plan->row_counter[grp];

  // log-scale set: slot g at fsm[g * 3 .. + 3); linear-scale set behind it: slot g at
  // [Gt * 3 (if both) + g * 5 .. + 5).  Odd strides, so the slots of a warp spread over all 32
  // banks.  The spare slot Gt of a set (masked entries add 0 there) is the first slot of
  // whatever follows; the table ends with kSetWords spare words.
  AccCtx cx;
  {
    uint32_t sb = (uint32_t)__cvta_generic_to_shared(fsm);
    asm volatile("mov.u32 %0, %0;" : "+r"(sb));           // keep it in a register (no recomputation)
    cx.sb_log = sb;
    cx.sb_lin = sb + (LOG ? (uint32_t)Gt * (kLogWords * 4u) : 0u);
  }
  cx.mult_log = mult_log; cx.mult_lin = mult_lin; cx.g0 = g0; cx.last_slot = (uint32_t)(Gt - 1);
  cx.S1log = a.S1log; cx.S2log = a.S2log; cx.S1lin = a.S1lin; cx.S2lin = a.S2lin;
  const uint32_t sb_log = cx.sb_log, sb_lin = cx.sb_lin, last_slot = cx.last_slot;
  constexpr int kWordsPerGene = (LOG ? kLogWords : 0) + (LIN ? kSetWords : 0);
  for (int i = tid; i < kWordsPerGene * Gt + kSetWords; i += kFuThreads) fsm[i] = 0u;

  // Row grabs (lane 0 only holds the result).  s_rows counts the rows this CTA has taken; the
  // warp whose grab crosses a multiple of 2^check_shift checks the tables (bit 62 of the result).
  auto grab_issue = [&]() -> long long {
    long long r = 0;
    if (lane == 0) {
      const unsigned c = atomicAdd(&s_rows, (unsigned)kFuRowsPerGrab);
      r = (long long)atomicAdd(counter, (unsigned long long)kFuRowsPerGrab);
      if (((c ^ (c + (unsigned)kFuRowsPerGrab)) >> a.check_shift) != 0u) r |= kCheckBit;
    }
    return r;
  };
  // A gene's words leave the CTA as 64-bit adds to the global integer totals: every 32-bit
  // word goes to its own counter (no carries between counters, so plain fire-and-forget
  // atomics; a counter overflows only after 2^32 flushes) -- independent of the CTA order and
  // of the grid.
  auto to_global_log = [&](int g, uint32_t w0, uint32_t s0, uint32_t W) {
    unsigned long long* acc = a.acc_log + g;
    const size_t G64 = (size_t)a.n_cols;
    const uint32_t hi = W & ((1u << kLogCarryBit) - 1u);
    // S1: w0 and its carry count in one add; S2: s0 and the upper field of W
    atomicAdd(acc, ((unsigned long long)(W >> kLogCarryBit) << 32) | w0);
    if (s0) atomicAdd(acc + 2 * G64, (unsigned long long)s0);
    if (hi) atomicAdd(acc + 3 * G64, (unsigned long long)hi);
  };
  auto to_global_lin = [&](int g, uint32_t w0, uint32_t w1, uint32_t s0, uint32_t s1, uint32_t s2) {
    unsigned long long* acc = a.acc_lin + g;
    const size_t G64 = (size_t)a.n_cols;
    if (w0) atomicAdd(acc, (unsigned long long)w0);
    if (w1) atomicAdd(acc + G64, (unsigned long long)w1);
    if (s0) atomicAdd(acc + 2 * G64, (unsigned long long)s0);
    if (s1) atomicAdd(acc + 3 * G64, (unsigned long long)s1);
    if (s2) atomicAdd(acc + 4 * G64, (unsigned long long)s2);
  };
  // Table check by ONE warp while the others keep adding: a gene whose packed word W (log
  // set) or top word (linear set) is at least half full is moved to the global totals, word
  // by word with an atomic exchange.  Each word is an independent sum (a carry is computed by
  // the adder from the value ITS atomic returned), so exchanging a word to 0 between two
  // adds loses nothing.  Between two checks of a gene a CTA adds at most
  // 2^check_shift + (rows in flight) <= kMaxRowsBetweenChecks rows, i.e. less than half of any field.
  auto check_tables = [&]() {
    for (int s = lane; s < ng_genes; s += 32) {
      if (LOG) {
        uint32_t* w = fsm + (size_t)s * kLogWords;
        const uint32_t W = *reinterpret_cast<volatile uint32_t*>(w + 2);
        if (a.flush_all || (W & ((1u << kLogCarryBit) - 1u)) >= (1u << (kLogCarryBit - 1)) ||
            (W >> kLogCarryBit) >= kLogCarryHalf) {
          const uint32_t w0 = atomicExch(w, 0u), s0 = atomicExch(w + 1, 0u), Wx = atomicExch(w + 2, 0u);
          if (w0 | s0 | Wx) to_global_log(g0 + s, w0, s0, Wx);
        }
      }
      if (LIN) {
        uint32_t* w = fsm + (LOG ? (size_t)Gt * kLogWords : 0) + (size_t)s * kSetWords;
        const uint32_t w1 = *reinterpret_cast<volatile uint32_t*>(w + 1);
        const uint32_t s2 = *reinterpret_cast<volatile uint32_t*>(w + 4);
        if (a.flush_all || ((w1 | s2) >> 31) != 0u) {
          const uint32_t x0 = atomicExch(w, 0u), x1 = atomicExch(w + 1, 0u), y0 = atomicExch(w + 2, 0u),
                         y1 = atomicExch(w + 3, 0u), y2 = atomicExch(w + 4, 0u);
          if (x0 | x1 | y0 | y1 | y2) to_global_lin(g0 + s, x0, x1, y0, y1, y2);
        }
      }
    }
  };

  // One quad of 4 consecutive entries.  Straight-line code when every value is in the usual
  // range (x' >= 0.25 and one-word integers), else through quad_rare (two-word integers, or
  // entry by entry).
  // EDGE: only entries e0 + k in [0, len) belong to the segment; the others (a neighbouring
  // segment's) are neutralised by adding 0 to the spare slot Gt, so the code stays branch-free.
  auto quad = [&](auto edge_tag, const int4 jv, const float4 xv, float scale, int e0, int len) -> float4 {
    constexpr bool EDGE = decltype(edge_tag)::value;
    const int j[4] = {jv.x, jv.y, jv.z, jv.w};
    const float x[4] = {xv.x, xv.y, xv.z, xv.w};
    float xn[4], xl[4], tl[4], tn[4];
    bool valid[4];
    unsigned okw = 1u;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      valid[k] = !EDGE || (unsigned)(e0 + k) < (unsigned)len;
      xn[k] = MOM ? x[k] : __fmul_rn(x[k], scale);
      xl[k] = MOM ? x[k] : log1p_ge_quarter(xn[k]);
      // branch-free: one test of the four entries' window bits instead of short-circuit branches (3.257 -> 3.202 ms)
      unsigned okk = (MOM || (LOG && !LIN) || xn[k] >= 0.25f) ? 1u : 0u;   // log only: implied by the window test
      if (LOG) { tl[k] = xl[k] * mult_log; okk &= in_window_log(tl[k]) ? 1u : 0u; }
      if (LIN) { tn[k] = xn[k] * mult_lin; okk &= in_window(tn[k]) ? 1u : 0u; }
      okw &= okk | (valid[k] ? 0u : 1u);
    }
    const bool ok = okw != 0u;
    if (ok) {
      uint32_t so[4], so3[4], al[4], an[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t slot = valid[k] ? min((uint32_t)(j[k] - g0), last_slot) : (uint32_t)Gt;
        if (LIN) so[k] = slot * (kSetWords * 4u);
        if (LOG) so3[k] = slot * (kLogWords * 4u);
        if (LOG) al[k] = valid[k] ? __float2uint_rz(tl[k]) : 0u;
        if (LIN) an[k] = valid[k] ? __float2uint_rz(tn[k]) : 0u;
      }
      if (LOG) acc3_quad(sb_log, so3, al);
      if (LIN) acc_quad(sb_lin, so, an);
    } else {
      const uint32_t vm = (valid[0] ? 1u : 0u) | (valid[1] ? 2u : 0u) | (valid[2] ? 4u : 0u) |
                          (valid[3] ? 8u : 0u);
      return quad_rare<LOG, LIN, MOM>(cx, jv, xv, scale, vm, (uint32_t)Gt);
    }
    return make_float4(xl[0], xl[1], xl[2], xl[3]);
  };

  {
    if (tid == 0) s_rows = 0u;
    __syncthreads();
    // Grabs are pipelined two deep: while grab g is processed, the row range of grab g + 1 is
    // already known, its row metadata is loaded and its segments are prefetched into L2, and
    // the atomic for grab g + 2 is in flight -- no latency chain between grabs.
    auto load_meta = [&](long long g0row, int64_t& mb, int64_t& me, float& ms) {
      mb = 0; me = 0; ms = 1.0f;
      const long long row = g0row + lane;                 // lanes 0..RG-1: one row each
      if (lane < kFuRowsPerGrab && row < a.n_rows) {
        const uint32_t* sp = a.splits + (size_t)row * sstride;
        const int64_t rb = a.indptr[row];
        mb = rb + sp[s0i];
        me = rb + sp[s1i];
        if (!MOM) ms = cell_scale(a.target_sum, a.cell_total[row]);
      }
    };
    // L2 look-ahead.  The head of the NEXT segment (its first kFuHead = 512 entries: lanes 0..15,
    // one 128-byte line per lane and array) is requested when the current segment starts; a
    // segment longer than that requests its own later parts kFuDist entries ahead while it is
    // walked (lookahead_in, 512 entries every 4 steps).  The distance is short on purpose: a line
    // fetched too early is evicted before it is used and read twice from DRAM (config 5, rows of
    // up to 25 000 entries: whole segment ahead 5.00 ms, 1024 entries 3.37 ms with 22 % re-reads,
    // 512 entries 3.10 ms; 256 entries is too little: 3.17 ms, and cfg3 3.37 instead of 3.25).
    auto l2_prefetch = [&](int64_t mb, int64_t me, int ri) {
      const int64_t pb = __shfl_sync(0xffffffffu, mb, ri);
      const int64_t pe = __shfl_sync(0xffffffffu, me, ri);
      const int64_t pcap = (int64_t)(pb & ~31LL) + kFuHead;
      const int64_t pe2 = pe < pcap ? pe : pcap;
      for (int64_t p = (pb & ~31LL) + lane * 32; p < pe2; p += 32 * 32) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(a.indices + p));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(a.data + p));
      }
    };
    auto lookahead_in = [&](int64_t abeg, int span, int st) {  // st % 4 == 0: entries [st 128 + kFuDist, + 512) of this segment
      const int off = st * 128 + kFuDist + lane * 32;
      if (lane < 16 && off < span) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(a.indices + abeg + off));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(a.data + abeg + off));
      }
    };
    long long r0 = __shfl_sync(0xffffffffu, grab_issue(), 0) & ~kCheckBit;
    int64_t mbeg = 0, mend = 0;
    float mscale = 1.0f;
    if (r0 < a.n_rows) load_meta(r0, mbeg, mend, mscale);
    long long rnext = __shfl_sync(0xffffffffu, grab_issue(), 0) & ~kCheckBit;
    while (r0 < a.n_rows) {
      const long long pending = grab_issue();             // grab g + 2; consumed after this grab
      const bool next_ok = rnext < a.n_rows;
      int64_t nbeg = 0, nend = 0;
      float nscale = 1.0f;
      if (next_ok) load_meta(rnext, nbeg, nend, nscale);
      // The grab's segments are walked in steps of 32 quads (one per lane); the loads of step
      // i + 1 are issued before step i is computed (software pipeline, one step deep).  A step
      // is "interior" when all of its 32 quads lie wholly inside the segment: no masks at all.
      struct Seg { int64_t abeg; int head, len, nq; float scale; };
      auto seg_of = [&](int ri) -> Seg {                  // warp-uniform; ri < kFuRowsPerGrab
        const int64_t beg = __shfl_sync(0xffffffffu, mbeg, ri);
        const int64_t end = __shfl_sync(0xffffffffu, mend, ri);
        Seg s;
        s.scale = __shfl_sync(0xffffffffu, mscale, ri);
        s.abeg = beg & ~3LL;
        s.head = (int)(beg - s.abeg);
        s.len = end > beg ? (int)(end - beg) : 0;
        s.nq = s.len > 0 ? (s.head + s.len + 3) >> 2 : 0;
        return s;
      };
      auto interior = [&](const Seg& s, int st) -> bool {
        return (st > 0 || s.head == 0) && (st * 128 + 128 <= s.head + s.len);
      };
      // dp: this lane's quad of step st in the data array (a running pointer: one add per step instead of
      // rebuilding the 64-bit address from the step number: 3.139 -> 3.083 ms); the index array lies a fixed
      // distance away
      const ptrdiff_t idelta = reinterpret_cast<const char*>(a.indices) - reinterpret_cast<const char*>(a.data);
      auto idx_of = [&](const float* dp) -> const int32_t* {
        return reinterpret_cast<const int32_t*>(reinterpret_cast<const char*>(dp) + idelta);
      };
      auto load_step = [&](const Seg& s, int st, const float* dp, int4& jv, float4& xv) {
        const int32_t* ip = idx_of(dp);
        if (interior(s, st)) {
          jv = __ldg(reinterpret_cast<const int4*>(ip));
          xv = *reinterpret_cast<const float4*>(dp);
        } else {
          const int q = st * 32 + lane;
          if (q < s.nq) {
            if ((dp - a.data) + 4 <= a.nnz) {
              jv = __ldg(reinterpret_cast<const int4*>(ip));
              xv = *reinterpret_cast<const float4*>(dp);
            } else {                                      // the last quad of the whole matrix
              const int e0 = q * 4 - s.head;
              jv = make_int4(0, 0, 0, 0);
              xv = make_float4(0.f, 0.f, 0.f, 0.f);
              if (e0 + 0 < s.len) { jv.x = __ldg(ip + 0); xv.x = dp[0]; }
              if (e0 + 1 < s.len) { jv.y = __ldg(ip + 1); xv.y = dp[1]; }
              if (e0 + 2 < s.len) { jv.z = __ldg(ip + 2); xv.z = dp[2]; }
            }
          }
        }
      };
      auto compute_step = [&](const Seg& s, int st, float* dq, const int4& jv, const float4& xv) {
        if (interior(s, st)) {
          const float4 r = quad(std::false_type{}, jv, xv, s.scale, 0, s.len);
          // x'' is written once and not read again by this pass: streaming stores (evict-first in L2) keep the
          // look-ahead's lines resident (3.257 -> 3.185 ms)
          if (!MOM) st_once(reinterpret_cast<float4*>(dq), r);
        } else {
          const int q = st * 32 + lane;
          const int e0 = q * 4 - s.head;
          if (q < s.nq) {
            const float4 r = quad(std::true_type{}, jv, xv, s.scale, e0, s.len);
            if (MOM) {
              // nothing is written back
            } else if (e0 >= 0 && e0 + 4 <= s.len) {
              *reinterpret_cast<float4*>(dq) = r;           // (plain: the line is shared with a neighbouring segment)
            } else {
              if ((unsigned)(e0 + 0) < (unsigned)s.len) dq[0] = r.x;
              if ((unsigned)(e0 + 1) < (unsigned)s.len) dq[1] = r.y;
              if ((unsigned)(e0 + 2) < (unsigned)s.len) dq[2] = r.z;
              if ((unsigned)(e0 + 3) < (unsigned)s.len) dq[3] = r.w;
            }
          }
        }
      };
      {
        Seg S;
        S.nq = 0;
        int ri = -1;
        while (++ri < kFuRowsPerGrab) { S = seg_of(ri); if (S.nq) break; }
        int4 jn = make_int4(0, 0, 0, 0);
        float4 xn4 = make_float4(0.f, 0.f, 0.f, 0.f);
        // kRun: the lane's quad address is carried from step to step (log-scale set: 3.139 -> 3.083 ms).  The
        // kernels with the linear-scale set have no register to spare for it (measured: +6 % / +9 % from
        // spills) and rebuild the address from the step number.
        constexpr bool kRun = LOG && !LIN;
        auto quad_ptr = [&](const Seg& s, int st) -> float* { return a.data + (s.abeg + 4 * (st * 32 + lane)); };
        float* dpc = a.data;
        if (ri < kFuRowsPerGrab) { dpc = quad_ptr(S, 0); load_step(S, 0, dpc, jn, xn4); }
        while (ri < kFuRowsPerGrab) {
          const int nsteps = (S.nq + 31) >> 5;
          int nri = ri;
          float* dpn = dpc;
          // the next row's segment (of this grab or the first of the next) goes to L2 now
          if (ri + 1 < kFuRowsPerGrab) l2_prefetch(mbeg, mend, ri + 1);
          else if (next_ok) l2_prefetch(nbeg, nend, 0);
#pragma unroll 1
          for (int st = 0; st < nsteps; ++st) {
            const int4 jc = jn;
            const float4 xc = xn4;
            if ((st & 3) == 0 && st * 128 + kFuDist < S.head + S.len) lookahead_in(S.abeg, S.head + S.len, st);
            if (st + 1 < nsteps) {
              load_step(S, st + 1, kRun ? dpc + 128 : quad_ptr(S, st + 1), jn, xn4);
            } else {                                      // prefetch the next segment's first step
              Seg N;
              N.nq = 0;
              while (++nri < kFuRowsPerGrab) { N = seg_of(nri); if (N.nq) break; }
              if (nri < kFuRowsPerGrab) { dpn = quad_ptr(N, 0); load_step(N, 0, dpn, jn, xn4); }
            }
            compute_step(S, st, kRun ? dpc : quad_ptr(S, st), jc, xc);
            if (kRun) dpc += 128;
          }
          if (kRun) dpc = dpn;
          ri = nri;
          if (ri < kFuRowsPerGrab) S = seg_of(ri);
        }
      }
      r0 = rnext; mbeg = nbeg; mend = nend; mscale = nscale;
      rnext = __shfl_sync(0xffffffffu, pending, 0);
      if (rnext & kCheckBit) { rnext &= ~kCheckBit; check_tables(); }
    }
    __syncthreads();
    // the matrix is exhausted: everything left in the tables goes to the global totals
    for (int s = tid; s < ng_genes; s += kFuThreads) {
      if (LOG) {
        const uint32_t* w = fsm + (size_t)s * kLogWords;
        if (w[0] | w[1] | w[2]) to_global_log(g0 + s, w[0], w[1], w[2]);
      }
      if (LIN) {
        const uint32_t* w = fsm + (LOG ? (size_t)Gt * kLogWords : 0) + (size_t)s * kSetWords;
        if (w[0] | w[1] | w[2] | w[3] | w[4]) to_global_lin(g0 + s, w[0], w[1], w[2], w[3], w[4]);
      }
    }
  }
}

template <bool LOG, bool LIN>
__global__ void __launch_bounds__(kFuThreads, 1) fused_stream_kernel(const FusedArgs a) {
  extern __shared__ __align__(16) uint32_t fsm[];
  __shared__ unsigned s_rows;
  fused_stream_body<LOG, LIN, false>(a, fsm, s_rows);
}

// rsc_gene_moments, transform 0 ("per-gene mean and variance, computed using a
// custom GPU reduction kernel that operates directly on sparse matrices"; L137): the same
// walk and accumulators with the normalise / log1p / store stage compiled out (8 B / nnz, read
// only).  The accumulator scheme was chosen on the device (moments_plan_kernel).
__global__ void __launch_bounds__(kFuThreads, 1) moments_stream_kernel(const FusedArgs a) {
  extern __shared__ __align__(16) uint32_t fsm[];
  __shared__ unsigned s_rows;
  if (a.plan->scheme == 1) fused_stream_body<true, false, true>(a, fsm, s_rows);
  else fused_stream_body<false, true, true>(a, fsm, s_rows);
}

// ------------------------------------------------------------------ double accumulators
// RSC_MOMENTS_FP64_ACC: per-gene doubles in shared memory, CAS atomics; any value range.
template <bool LOG, bool LIN>
__global__ void __launch_bounds__(kFuThreads, 1) fused_stream_fp64_kernel(const FusedArgs a) {
  extern __shared__ __align__(16) uint32_t fsm[];
  __shared__ unsigned s_rows;
  const int tid = threadIdx.x, lane = tid & 31;
  const int Gt = a.Gt;
  const int K = a.n_fine;
  const FusedPlan* plan = a.plan;
  int grp = 0;
  {
    const int ng = plan->n_groups;
    while (grp + 1 < ng && (int)blockIdx.x >= plan->cta_first[grp + 1]) ++grp;
  }
  const int f0 = (grp * K) / plan->n_groups;              // group = blocks [grp K / ng, (grp + 1) K / ng)
  const int f1 = ((grp + 1) * K) / plan->n_groups;
  const int g0 = f0 << RSC_SPLIT_SHIFT;
  const int ng_genes = min(a.n_cols, f1 << RSC_SPLIT_SHIFT) - g0;
  unsigned long long* counter = &a.plan->row_counter[grp];
  double* tlog = reinterpret_cast<double*>(fsm);                    // [2][Gt]
  double* tlin = tlog + (LOG ? 2 * (size_t)Gt : 0);                 // [2][Gt]
  constexpr int kSets = (LOG ? 1 : 0) + (LIN ? 1 : 0);
  for (int i = tid; i < kSets * 2 * Gt; i += kFuThreads) tlog[i] = 0.0;

  int done;
  do {
    if (tid == 0) s_rows = 0u;
    __syncthreads();
    int saw_end = 0;
    for (;;) {
      long long r0 = -1;
      if (lane == 0) {
        const unsigned c = atomicAdd(&s_rows, (unsigned)kFuRowsPerGrab);
        if (c < a.row_budget) r0 = (long long)atomicAdd(counter, (unsigned long long)kFuRowsPerGrab);
      }
      r0 = __shfl_sync(0xffffffffu, r0, 0);
      if (r0 < 0) break;
      if (r0 >= a.n_rows) { saw_end = 1; break; }
      const int nr = (int)min((long long)kFuRowsPerGrab, a.n_rows - r0);
      for (int ri = 0; ri < nr; ++ri) {
        const long long row = r0 + ri;
        const uint32_t* sp = a.splits + (size_t)row * (size_t)(K + 1);
        const int64_t rb = a.indptr[row];
        const int64_t beg = rb + sp[f0], end = rb + sp[f1];
        const float scale = cell_scale(a.target_sum, a.cell_total[row]);
        for (int64_t p = beg + lane; p < end; p += 32) {
          const int slot = __ldg(a.indices + p) - g0;
          const float xn = __fmul_rn(a.data[p], scale);
          const float xl = log1p_f32(xn);
          a.data[p] = xl;
          if ((unsigned)slot >= (unsigned)Gt) continue;
          if (LOG) { const double v = (double)xl; atomicAdd(tlog + slot, v); atomicAdd(tlog + Gt + slot, v * v); }
          if (LIN) { const double v = (double)xn; atomicAdd(tlin + slot, v); atomicAdd(tlin + Gt + slot, v * v); }
        }
      }
    }
    done = __syncthreads_or(saw_end);
    for (int s = tid; s < ng_genes; s += kFuThreads) {
      const int g = g0 + s;
      if (LOG && (tlog[s] != 0.0 || tlog[Gt + s] != 0.0)) {
        atomicAdd(&a.S1log[g], tlog[s]); atomicAdd(&a.S2log[g], tlog[Gt + s]);
        tlog[s] = 0.0; tlog[Gt + s] = 0.0;
      }
      if (LIN && (tlin[s] != 0.0 || tlin[Gt + s] != 0.0)) {
        atomicAdd(&a.S1lin[g], tlin[s]); atomicAdd(&a.S2lin[g], tlin[Gt + s]);
        tlin[s] = 0.0; tlin[Gt + s] = 0.0;
      }
    }
  } while (!done);
}

// ------------------------------------------------------------------ integer totals -> sums, moments
// S += total * 2^-k (S holds what the out-of-window values added directly, usually 0), then
// mean = S1 / n, var = max(0, (S2 - n mean^2) / (n - ddof)) as rsc_moments_finalize
__global__ void __launch_bounds__(256)
fused_finish_kernel(int G, double n, double denom, const FusedPlan* __restrict__ plan, int is_lin,
                    const unsigned long long* __restrict__ acc, double* __restrict__ S1,
                    double* __restrict__ S2, double* __restrict__ mean, double* __restrict__ var) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= G) return;
  if (is_lin < 0) is_lin = plan->scheme == 2;            // moments-only pass: the scheme the plan chose
  const MomentScale sc = is_lin ? plan->sc_lin : plan->sc_log;
  const double two32 = 4294967296.0;
  const size_t Gs = (size_t)G;
  const double t1 = (double)acc[Gs + g] * two32 + (double)acc[g];
  const double t2 = ((double)acc[4 * Gs + g] * two32 + (double)acc[3 * Gs + g]) * two32 + (double)acc[2 * Gs + g];
  const double s1 = S1[g] + t1 * sc.inv1, s2 = S2[g] + t2 * sc.inv2;
  S1[g] = s1;
  S2[g] = s2;
  const double m = s1 / n;
  const double v = (s2 - n * m * m) / denom;
  if (mean) mean[g] = m;
  if (var) var[g] = v > 0.0 ? v : (v == v ? 0.0 : v);
}

// the integer totals of one set -> S1 / S2 / mean / var (also used by single.cu)
int launch_fused_finish(int32_t G, int64_t n_rows, int ddof, const FusedPlan* plan, int is_lin,
                        const unsigned long long* acc, double* S1, double* S2, double* mean, double* var,
                        cudaStream_t st) {
  const unsigned blocks = (unsigned)(((size_t)G + 255) / 256);
  fused_finish_kernel<<<blocks, 256, 0, st>>>(G, (double)n_rows, (double)(n_rows - ddof), plan, is_lin, acc, S1, S2,
                                              mean, var);
  RSC_LAUNCH_CHECK("fused_finish_kernel");
  return RSC_OK;
}

// ------------------------------------------------------------------ host side
int launch_fused_generic(const rsc_csr&, float, const int64_t*, int, double*, double*, double*,
                         double*, cudaStream_t);

static int fused_grid() { return g_opt.grid_ctas.load() > 0 ? g_opt.grid_ctas.load() : sm_count(); }

// bytes of shared-memory accumulators per gene
static int bytes_per_gene(int which) {
  const int sets = ((which & RSC_MOMENTS_LOG) ? 1 : 0) + ((which & RSC_MOMENTS_LIN) ? 1 : 0);
  if (which & RSC_MOMENTS_FP64_ACC) return sets * 16;
  return ((which & RSC_MOMENTS_LOG) ? kLogWords * 4 : 0) + ((which & RSC_MOMENTS_LIN) ? kSetWords * 4 : 0);
}

// column blocks per group: as many as fit, then evened out over the groups
static int fine_per_group(int32_t n_cols, int which) {
  const int bpg = bytes_per_gene(which);
  if (bpg == 0) return 0;
  const int fit = (int)((kMaxDynSmem - 64) / ((size_t)bpg * RSC_SPLIT_WIDTH));
  if (fit < 1) return 0;
  const int K = split_blocks(n_cols);
  const int ng = (K + fit - 1) / fit;
  return (K + ng - 1) / ng;
}

// true when the streaming kernel can serve this call (else: generic L2-atomic kernel)
static bool fused_fast_ok(const rsc_csr& X, int which) {
  if (!(X.flags & RSC_CSR_SORTED) || g_opt.force_generic) return false;
  if ((which & 3) == 0) return false;
  // 128-bit accesses need 16-byte aligned arrays
  if ((reinterpret_cast<uintptr_t>(X.indices) | reinterpret_cast<uintptr_t>(X.data)) & 15) return false;
  const int fpg = fine_per_group(X.n_cols, which);
  if (fpg < 1) return false;
  const int K = split_blocks(X.n_cols);
  const int ng = (K + fpg - 1) / fpg;
  return ng <= kMaxGroups && ng <= fused_grid();
}

// the row split entries the streaming kernel reads: the edges (c K) / ng of its groups
int fused_split_blocks(int32_t n_cols, int which, int32_t* out, int32_t cap) {
  const int fpg = fine_per_group(n_cols, which);
  if (fpg < 1 || (which & 3) == 0) return 0;
  const int K = split_blocks(n_cols);
  const int ng = (K + fpg - 1) / fpg;
  if (ng + 1 > cap) return ng + 1;
  for (int c = 0; c <= ng; ++c) out[c] = (c * K) / ng;
  return ng + 1;
}

size_t fused_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t) {
  const size_t K1 = (size_t)split_blocks(n_cols) + 1;
  return 4 * align_up(sizeof(double) * (size_t)n_cols, 256) + align_up(sizeof(FusedPlan), 256) +
         align_up(sizeof(uint32_t) * (size_t)n_rows * K1, 256) +
         2 * align_up(5 * sizeof(unsigned long long) * (size_t)n_cols, 256);
}

template <typename Kern>
static int launch_stream(Kern kern, const FusedArgs& a, size_t smem, cudaStream_t st) {
  RSC_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem));
  kern<<<fused_grid(), kFuThreads, smem, st>>>(a);
  RSC_LAUNCH_CHECK("fused_stream_kernel");
  return RSC_OK;
}

int launch_fused(const rsc_csr& X, float target_sum, const int64_t* cell_total_i64,
                 const int32_t* gene_n_cells, const uint32_t* row_splits, int which, int ddof,
                 double* mean_log, double* var_log, double* mean_lin, double* var_lin,
                 double* sums_out, void* ws, size_t, cudaStream_t st) {
  const size_t gsz = align_up(sizeof(double) * (size_t)X.n_cols, 256);
  unsigned char* w = static_cast<unsigned char*>(ws);
  const size_t G = (size_t)X.n_cols;
  double* S1log = sums_out ? sums_out : reinterpret_cast<double*>(w);
  double* S2log = sums_out ? sums_out + G : reinterpret_cast<double*>(w + gsz);
  double* S1lin = sums_out ? sums_out + 2 * G : reinterpret_cast<double*>(w + 2 * gsz);
  double* S2lin = sums_out ? sums_out + 3 * G : reinterpret_cast<double*>(w + 3 * gsz);
  int rc;
  if (!fused_fast_ok(X, which) || X.n_rows == 0) {
    rc = launch_fused_generic(X, target_sum, cell_total_i64, which, S1log, S2log, S1lin, S2lin, st);
    if (rc != RSC_OK) return rc;
  } else {
    // workspace: 4 double sums | 2 x 5 integer totals | plan | (row split table); the sums, the
    // totals and the plan (tmax) start from zero: one memset when the sums live in the workspace
    const size_t asz = align_up(5 * sizeof(unsigned long long) * G, 256);
    unsigned char* accb = w + 4 * gsz;
    FusedPlan* plan = reinterpret_cast<FusedPlan*>(accb + 2 * asz);
    if (sums_out == nullptr) {
      RSC_CUDA(cudaMemsetAsync(w, 0, 4 * gsz + 2 * asz + sizeof(FusedPlan), st));
    } else {
      // only the requested sets are written (rsc.h): a caller may keep another set's sums here
      if (which & RSC_MOMENTS_LOG) RSC_CUDA(cudaMemsetAsync(sums_out, 0, 2 * sizeof(double) * G, st));
      if (which & RSC_MOMENTS_LIN) RSC_CUDA(cudaMemsetAsync(sums_out + 2 * G, 0, 2 * sizeof(double) * G, st));
      RSC_CUDA(cudaMemsetAsync(accb, 0, 2 * asz + sizeof(FusedPlan), st));
    }
    if (row_splits == nullptr) {
      uint32_t* sp = reinterpret_cast<uint32_t*>(accb + 2 * asz + align_up(sizeof(FusedPlan), 256));
      if ((rc = launch_row_splits(X, sp, st)) != RSC_OK) return rc;
      row_splits = sp;
    }
    FusedArgs a;
    a.n_rows = X.n_rows; a.n_cols = X.n_cols; a.nnz = X.nnz; a.n_fine = split_blocks(X.n_cols);
    a.fine_per_group = fine_per_group(X.n_cols, which);
    a.Gt = a.fine_per_group * RSC_SPLIT_WIDTH;
    a.indptr = X.indptr; a.indices = X.indices; a.data = X.data; a.cell_total = cell_total_i64;
    a.splits = row_splits; a.target_sum = target_sum;
    a.row_budget = 4000u;
    a.check_shift = 0u;                                         // largest power of two <= the option (<= 512)
    while ((2u << a.check_shift) <= (uint32_t)kCheckRows && (2u << a.check_shift) <= (uint32_t)g_opt.fused_row_budget) ++a.check_shift;
    a.flush_all = g_opt.flush_all ? 1u : 0u;
    a.S1log = S1log; a.S2log = S2log; a.S1lin = S1lin; a.S2lin = S2lin; a.plan = plan;
    const bool int_acc = !(which & RSC_MOMENTS_FP64_ACC);
    a.acc_log = reinterpret_cast<unsigned long long*>(accb);
    a.acc_lin = reinterpret_cast<unsigned long long*>(accb + asz);
    if (!(which & RSC_MOMENTS_FP64_ACC)) {
      // cell depths place the windows: the largest total (linear scale), the binades of the
      // cells' smallest x'' (log scale)
      int64_t blocks = (X.n_rows + 255) / 256;
      const int64_t cap = (int64_t)sm_count() * 4;
      if (blocks > cap) blocks = cap;
      fused_tmax_kernel<<<(unsigned)blocks, 256, 0, st>>>(plan, X.n_rows, cell_total_i64, target_sum);
      RSC_LAUNCH_CHECK("fused_tmax_kernel");
    }
    fused_plan_kernel<<<1, 1024, 0, st>>>(plan, X.n_cols, a.n_fine, a.fine_per_group, fused_grid(),
                                          target_sum, (long long)X.n_rows, gene_n_cells);
    RSC_LAUNCH_CHECK("fused_plan_kernel");
    const size_t smem = (size_t)bytes_per_gene(which) * (size_t)a.Gt + 32;   // + the spare slot
    switch (which & 7) {
      case 1: rc = launch_stream(fused_stream_kernel<true, false>, a, smem, st); break;
      case 2: rc = launch_stream(fused_stream_kernel<false, true>, a, smem, st); break;
      case 3: rc = launch_stream(fused_stream_kernel<true, true>, a, smem, st); break;
      case 5: rc = launch_stream(fused_stream_fp64_kernel<true, false>, a, smem, st); break;
      case 6: rc = launch_stream(fused_stream_fp64_kernel<false, true>, a, smem, st); break;
      default: rc = launch_stream(fused_stream_fp64_kernel<true, true>, a, smem, st); break;
    }
    if (rc != RSC_OK) return rc;
    if (int_acc) {
      const unsigned blocks = (unsigned)((G + 255) / 256);
      const double n = (double)X.n_rows, denom = (double)(X.n_rows - ddof);
      if (which & RSC_MOMENTS_LOG) {
        fused_finish_kernel<<<blocks, 256, 0, st>>>(X.n_cols, n, denom, plan, 0, a.acc_log, S1log, S2log,
                                                    mean_log, var_log);
        RSC_LAUNCH_CHECK("fused_finish_kernel");
      }
      if (which & RSC_MOMENTS_LIN) {
        fused_finish_kernel<<<blocks, 256, 0, st>>>(X.n_cols, n, denom, plan, 1, a.acc_lin, S1lin, S2lin,
                                                    mean_lin, var_lin);
        RSC_LAUNCH_CHECK("fused_finish_kernel");
      }
      return RSC_OK;
    }
  }
  if (which & RSC_MOMENTS_LOG) {
    rc = finalize_moments(X.n_cols, X.n_rows, ddof, S1log, S2log, mean_log, var_log, st);
    if (rc != RSC_OK) return rc;
  }
  if (which & RSC_MOMENTS_LIN) {
    rc = finalize_moments(X.n_cols, X.n_rows, ddof, S1lin, S2lin, mean_lin, var_lin, st);
    if (rc != RSC_OK) return rc;
  }
  return RSC_OK;
}

// ------------------------------------------------------------------ rsc_gene_moments, fast path
size_t moments_fast_workspace_bytes(int64_t n_rows, int32_t n_cols) {
  return 2 * align_up(sizeof(double) * (size_t)n_cols, 256) +
         align_up(5 * sizeof(unsigned long long) * (size_t)n_cols, 256) + align_up(sizeof(FusedPlan), 256) +
         align_up(sizeof(uint32_t) * (size_t)(n_rows > 0 ? n_rows : 0) * kNeedStride, 256);
}

// sorted rows, 16-byte aligned arrays, at most kNeedStride - 1 groups in the worst (five-word) case
bool moments_fast_ok(const rsc_csr& X) {
  if (!(X.flags & RSC_CSR_SORTED) || g_opt.force_generic || X.n_rows == 0 || X.nnz == 0) return false;
  if ((reinterpret_cast<uintptr_t>(X.indices) | reinterpret_cast<uintptr_t>(X.data)) & 15) return false;
  const int fit = (int)((kMaxDynSmem - 64) / ((size_t)kSetWords * 4 * RSC_SPLIT_WIDTH));
  const int K = split_blocks(X.n_cols);
  const int ng = (K + fit - 1) / fit;
  return ng <= kNeedStride - 1 && ng <= fused_grid();
}

int launch_moments_fast(const rsc_csr& X, int ddof, double* mean, double* var, double* sum, double* sumsq,
                        void* ws, cudaStream_t st) {
  const size_t G = (size_t)X.n_cols;
  const size_t gsz = align_up(sizeof(double) * G, 256);
  const size_t asz = align_up(5 * sizeof(unsigned long long) * G, 256);
  unsigned char* w = static_cast<unsigned char*>(ws);
  double* S1 = sum ? sum : reinterpret_cast<double*>(w);
  double* S2 = sumsq ? sumsq : reinterpret_cast<double*>(w + gsz);
  unsigned char* accb = w + 2 * gsz;
  FusedPlan* plan = reinterpret_cast<FusedPlan*>(accb + asz);
  uint32_t* splits = reinterpret_cast<uint32_t*>(accb + asz + align_up(sizeof(FusedPlan), 256));
  RSC_CUDA(cudaMemsetAsync(S1, 0, sizeof(double) * G, st));
  RSC_CUDA(cudaMemsetAsync(S2, 0, sizeof(double) * G, st));
  RSC_CUDA(cudaMemsetAsync(accb, 0, asz + sizeof(FusedPlan), st));
  const int K = split_blocks(X.n_cols);
  moments_plan_kernel<<<1, 1024, 0, st>>>(plan, X.n_cols, K, fused_grid(), (long long)X.n_rows,
                                          (long long)X.nnz, X.indices, X.data);
  RSC_LAUNCH_CHECK("moments_plan_kernel");
  row_splits_compact_kernel<<<(unsigned)((X.n_rows + 255) / 256), 256, 0, st>>>(X.n_rows, X.n_cols, X.indptr,
                                                                              X.indices, plan, splits);
  RSC_LAUNCH_CHECK("row_splits_compact_kernel");
  FusedArgs a;
  a.n_rows = X.n_rows; a.n_cols = X.n_cols; a.nnz = X.nnz; a.n_fine = K;
  a.fine_per_group = 0; a.Gt = 0;                               // from the plan
  a.indptr = X.indptr; a.indices = X.indices; a.data = X.data; a.cell_total = nullptr;
  a.splits = splits; a.target_sum = 1.0f; a.row_budget = 0u;
  a.check_shift = 0u;
  while ((2u << a.check_shift) <= (uint32_t)kCheckRows && (2u << a.check_shift) <= (uint32_t)g_opt.fused_row_budget) ++a.check_shift;
  a.flush_all = g_opt.flush_all ? 1u : 0u;
  a.S1log = S1; a.S2log = S2; a.S1lin = S1; a.S2lin = S2; a.plan = plan;
  a.acc_log = reinterpret_cast<unsigned long long*>(accb);
  a.acc_lin = a.acc_log;
  RSC_CUDA(cudaFuncSetAttribute(moments_stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kMaxDynSmem));
  moments_stream_kernel<<<fused_grid(), kFuThreads, kMaxDynSmem, st>>>(a);
  RSC_LAUNCH_CHECK("moments_stream_kernel");
  fused_finish_kernel<<<(unsigned)((G + 255) / 256), 256, 0, st>>>(
      X.n_cols, (double)X.n_rows, (double)(X.n_rows - ddof), plan, -1, a.acc_log, S1, S2, mean, var);
  RSC_LAUNCH_CHECK("fused_finish_kernel");
  return RSC_OK;
}

}  // namespace rsc
