// rsc_normalize_log1p_moments, streaming kernel: x' = x * scale_i, x'' = log1p(x') written
// back, per-gene sums of x'' / x''^2 (log scale) and x' / x'^2 (linear scale) accumulated on
// chip.  PAPER.md:L91 (normalize_total, log1p, "per-gene mean and variance, computed using a
// custom GPU reduction kernel that operates directly on sparse matrices"), L137; the fusion
// itself is BASELINE.json north_star's, not the paper's.  12 B / nnz of DRAM traffic.
//
// Design:
//   * Gene-range groups.  G genes x 4..5 64-bit accumulators do not fit one SM's shared
//     memory, so the columns are cut into groups of `fine_per_group` blocks of
//     RSC_SPLIT_WIDTH genes; a CTA serves ONE group and keeps that group's accumulators
//     (<= 227 KB) private.  Rows are sorted, so a group's entries are one contiguous
//     segment of every row, located through the row split table (written by the QC pass or
//     by row_splits_kernel).  CTAs are dealt to groups in proportion to the groups' nnz
//     (fused_plan_kernel, on the device), rows to a group's CTAs by an atomic cursor.
//   * Accumulators.  Default: 64-bit FIXED-POINT sums held as two u32 words and updated
//     with two native 32-bit shared atomics (ATOMS.ADD; the low word's carry-out is added
//     to the high word), because 64-bit / floating-point shared atomics are CAS loops on
//     sm_100 (5x slower, measured).  Integer adds commute, so the sums are independent of
//     the order of the adds.  Scales are powers of two chosen from target_sum so that
//     4096 rows cannot overflow; a CTA flushes to the global double sums after at most
//     4096 rows.  Resolution: 2^-48 (S1 log), 2^-44 (S2 log), 2^(E-52) (S1 lin, 2^E >
//     target_sum); S2 lin uses two windows (x' < 2^(E-10): 2^(2E-72), else 2^(2E-52)), so
//     every addend keeps >= 31 significant bits.  RSC_MOMENTS_FP64_ACC selects plain
//     double accumulators (CAS atomics) instead: any value range, slower.
#include <math.h>

#include "common.cuh"

namespace rsc {

constexpr int kFuThreads = 1024;
constexpr int kFuUnroll = 4;
constexpr int kFuRowsPerGrab = 4;
constexpr int kMaxGroups = 64;

struct FusedPlan {            // in the workspace; written by fused_plan_kernel
  int32_t n_groups;
  int32_t pad;
  int32_t cta_first[kMaxGroups + 1];
  unsigned long long row_counter[kMaxGroups];
};

struct FixedScales {
  float m_s1log, m_s2log_h, m_s1lin, m_s2hi_h, m_s2lo_h, lin_theta;
  double inv_s1log, inv_s2log, inv_s1lin, inv_s2hi, inv_s2lo;
};

struct FusedArgs {
  int64_t n_rows;
  int32_t n_cols;
  int32_t n_fine;            // K
  int32_t fine_per_group;
  int32_t Gt;                // accumulator slots per CTA = fine_per_group * RSC_SPLIT_WIDTH
  const int64_t* indptr;
  const int32_t* indices;
  float* data;
  const int64_t* cell_total;
  const uint32_t* splits;
  float target_sum;
  uint32_t row_budget;       // a CTA stops grabbing rows once it has taken this many (then flushes)
  FixedScales fs;
  double* S1log; double* S2log; double* S1lin; double* S2lin;
  FusedPlan* plan;
};

// ------------------------------------------------------------------ plan (1 CTA)
__global__ void __launch_bounds__(1024)
fused_plan_kernel(FusedPlan* plan, int G, int K, int fine_per_group, int grid,
                  const int32_t* __restrict__ gene_n_cells) {
  __shared__ double mass[kMaxGroups];
  const int tid = threadIdx.x;
  const int ng = (K + fine_per_group - 1) / fine_per_group;
  if (tid < kMaxGroups) mass[tid] = 0.0;
  __syncthreads();
  const int gw = fine_per_group << RSC_SPLIT_SHIFT;       // genes per group
  for (int c = 0; c < ng; ++c) {
    const int g0 = c * gw, g1 = min(G, g0 + gw);
    double m = 0.0;
    for (int g = g0 + tid; g < g1; g += 1024) {
      const int v = gene_n_cells ? gene_n_cells[g] : 1;
      m += (double)(v > 0 ? v : 0);
    }
    m = warp_sum(m);
    if ((tid & 31) == 0 && m != 0.0) atomicAdd(&mass[c], m);
  }
  __syncthreads();
  if (tid == 0) {
    double total = 0.0;
    for (int c = 0; c < ng; ++c) total += mass[c];
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
}

// ------------------------------------------------------------------ accumulator primitives
// 64-bit add on two u32 words with native shared atomics; exact modulo 2^64 for any
// interleaving (the carry of the low word is added to the high word by whoever caused it).
__device__ __forceinline__ void add64(uint32_t* lo, uint32_t* hi, unsigned long long v) {
  const uint32_t vl = (uint32_t)v, vh = (uint32_t)(v >> 32);
  const uint32_t old = atomicAdd(lo, vl);
  atomicAdd(hi, vh + ((old + vl) < old ? 1u : 0u));
}

template <bool LOG, bool LIN, bool FIXED>
struct Acc {
  static constexpr int kLogWords = LOG ? (FIXED ? 4 : 4) : 0;     // u32 words per gene
  static constexpr int kLinWords = LIN ? (FIXED ? 6 : 4) : 0;
  static constexpr int kWords = kLogWords + kLinWords;
};

template <bool LOG, bool LIN, bool FIXED>
__global__ void __launch_bounds__(kFuThreads, 1) fused_stream_kernel(const FusedArgs a) {
  extern __shared__ __align__(16) uint32_t fsm[];
  using A = Acc<LOG, LIN, FIXED>;
  __shared__ unsigned s_rows;
  const int tid = threadIdx.x, lane = tid & 31;
  const int Gt = a.Gt;
  const int K = a.n_fine;

  // which group does this CTA serve?
  const FusedPlan* plan = a.plan;
  int grp = 0;
  {
    const int ng = plan->n_groups;
    while (grp + 1 < ng && (int)blockIdx.x >= plan->cta_first[grp + 1]) ++grp;
  }
  const int f0 = grp * a.fine_per_group;
  const int f1 = min(K, f0 + a.fine_per_group);
  const int g0 = f0 << RSC_SPLIT_SHIFT;
  const int ng_genes = min(a.n_cols, f1 << RSC_SPLIT_SHIFT) - g0;
  unsigned long long* counter = &a.plan->row_counter[grp];

  uint32_t* wlog = fsm;                                   // LOG words: [4][Gt]
  uint32_t* wlin = fsm + (size_t)A::kLogWords * Gt;       // LIN words: [6 or 4][Gt]
  for (int i = tid; i < A::kWords * Gt; i += kFuThreads) fsm[i] = 0u;

  const FixedScales fs = a.fs;

  auto grab_issue = [&]() -> long long {                  // lane 0 only holds the result
    long long r = -1;
    if (lane == 0) {
      const unsigned c = atomicAdd(&s_rows, (unsigned)kFuRowsPerGrab);
      if (c < a.row_budget) r = (long long)atomicAdd(counter, (unsigned long long)kFuRowsPerGrab);
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
      const long long pending = grab_issue();             // consumed after this batch of rows
      // lanes 0..RG-1 fetch the segment bounds and the scale of one row each
      int64_t mbeg = 0, mend = 0;
      float mscale = 1.0f;
      {
        const long long row = r0 + lane;
        if (lane < kFuRowsPerGrab && row < a.n_rows) {
          const uint32_t* sp = a.splits + (size_t)row * (size_t)(K + 1);
          const int64_t rb = a.indptr[row];
          mbeg = rb + sp[f0];
          mend = rb + sp[f1];
          mscale = cell_scale(a.target_sum, a.cell_total[row]);
        }
      }
#pragma unroll 1
      for (int ri = 0; ri < kFuRowsPerGrab; ++ri) {
        const int64_t beg = __shfl_sync(0xffffffffu, mbeg, ri);
        const int64_t end = __shfl_sync(0xffffffffu, mend, ri);
        const float scale = __shfl_sync(0xffffffffu, mscale, ri);
        for (int64_t base = beg; base < end; base += 32 * kFuUnroll) {
          int j[kFuUnroll];
          float x[kFuUnroll];
#pragma unroll
          for (int u = 0; u < kFuUnroll; ++u) {
            const int64_t p = base + u * 32 + lane;
            const bool ok = p < end;
            j[u] = ok ? __ldg(a.indices + p) : -1;
            x[u] = ok ? a.data[p] : 0.0f;
          }
#pragma unroll
          for (int u = 0; u < kFuUnroll; ++u) {
            const int slot = j[u] - g0;
            if (j[u] >= 0 && (unsigned)slot < (unsigned)Gt) {
              const float xn = __fmul_rn(x[u], scale);
              const float xl = log1p_f32(xn);
              a.data[base + u * 32 + lane] = xl;
              if (FIXED) {
                if (LOG) {
                  add64(wlog + slot, wlog + Gt + slot, __float2ull_rn(xl * fs.m_s1log));
                  const double d = (double)(xl * fs.m_s2log_h);
                  add64(wlog + 2 * Gt + slot, wlog + 3 * Gt + slot, __double2ull_rn(d * d));
                }
                if (LIN) {
                  add64(wlin + slot, wlin + Gt + slot, __float2ull_rn(xn * fs.m_s1lin));
                  const bool small = xn < fs.lin_theta;
                  const double d = (double)(xn * (small ? fs.m_s2lo_h : fs.m_s2hi_h));
                  uint32_t* w = wlin + (small ? 4 : 2) * Gt + slot;
                  add64(w, w + Gt, __double2ull_rn(d * d));
                }
              } else {
                if (LOG) {
                  double* t = reinterpret_cast<double*>(wlog);
                  const double v = (double)xl;
                  atomicAdd(t + slot, v);
                  atomicAdd(t + Gt + slot, v * v);
                }
                if (LIN) {
                  double* t = reinterpret_cast<double*>(wlin);
                  const double v = (double)xn;
                  atomicAdd(t + slot, v);
                  atomicAdd(t + Gt + slot, v * v);
                }
              }
            }
          }
        }
      }
      r0 = __shfl_sync(0xffffffffu, pending, 0);
    }
    done = __syncthreads_or(saw_end);
    // flush this CTA's accumulators into the global double sums and clear them
    for (int s = tid; s < ng_genes; s += kFuThreads) {
      const int g = g0 + s;
      if (FIXED) {
        if (LOG) {
          const unsigned long long v1 = ((unsigned long long)wlog[Gt + s] << 32) | wlog[s];
          const unsigned long long v2 = ((unsigned long long)wlog[3 * Gt + s] << 32) | wlog[2 * Gt + s];
          if (v1 | v2) {
            atomicAdd(&a.S1log[g], (double)v1 * fs.inv_s1log);
            atomicAdd(&a.S2log[g], (double)v2 * fs.inv_s2log);
            wlog[s] = 0u; wlog[Gt + s] = 0u; wlog[2 * Gt + s] = 0u; wlog[3 * Gt + s] = 0u;
          }
        }
        if (LIN) {
          const unsigned long long v1 = ((unsigned long long)wlin[Gt + s] << 32) | wlin[s];
          const unsigned long long vh = ((unsigned long long)wlin[3 * Gt + s] << 32) | wlin[2 * Gt + s];
          const unsigned long long vl = ((unsigned long long)wlin[5 * Gt + s] << 32) | wlin[4 * Gt + s];
          if (v1 | vh | vl) {
            atomicAdd(&a.S1lin[g], (double)v1 * fs.inv_s1lin);
            atomicAdd(&a.S2lin[g], (double)vh * fs.inv_s2hi + (double)vl * fs.inv_s2lo);
            wlin[s] = 0u; wlin[Gt + s] = 0u; wlin[2 * Gt + s] = 0u; wlin[3 * Gt + s] = 0u;
            wlin[4 * Gt + s] = 0u; wlin[5 * Gt + s] = 0u;
          }
        }
      } else {
        if (LOG) {
          double* t = reinterpret_cast<double*>(wlog);
          if (t[s] != 0.0 || t[Gt + s] != 0.0) {
            atomicAdd(&a.S1log[g], t[s]); atomicAdd(&a.S2log[g], t[Gt + s]);
            t[s] = 0.0; t[Gt + s] = 0.0;
          }
        }
        if (LIN) {
          double* t = reinterpret_cast<double*>(wlin);
          if (t[s] != 0.0 || t[Gt + s] != 0.0) {
            atomicAdd(&a.S1lin[g], t[s]); atomicAdd(&a.S2lin[g], t[Gt + s]);
            t[s] = 0.0; t[Gt + s] = 0.0;
          }
        }
      }
    }
  } while (!done);
}

// ------------------------------------------------------------------ host side
int launch_fused_generic(const rsc_csr&, float, const int64_t*, int, double*, double*, double*,
                         double*, cudaStream_t);

static int fused_grid() { return g_opt.grid_ctas > 0 ? g_opt.grid_ctas : sm_count(); }

static int words_per_gene(int which, bool fixed) {
  int w = 0;
  if (which & RSC_MOMENTS_LOG) w += 4;
  if (which & RSC_MOMENTS_LIN) w += fixed ? 6 : 4;
  return w;
}

// true when the streaming kernel can serve this call (else: generic L2-atomic kernel)
static bool fused_fast_ok(const rsc_csr& X, float target_sum, int which) {
  if (!(X.flags & RSC_CSR_SORTED) || g_opt.force_generic) return false;
  if ((which & 3) == 0) return false;
  const bool fixed = !(which & RSC_MOMENTS_FP64_ACC);
  if (fixed && !(target_sum < 1.0e9f)) return false;
  const int wpg = words_per_gene(which, fixed);
  const int fpg = (int)((kMaxDynSmem - 64) / ((size_t)wpg * 4 * RSC_SPLIT_WIDTH));
  if (fpg < 1) return false;
  const int K = split_blocks(X.n_cols);
  const int ng = (K + fpg - 1) / fpg;
  return ng <= kMaxGroups && ng <= fused_grid();
}

size_t fused_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t) {
  const size_t K1 = (size_t)split_blocks(n_cols) + 1;
  return 4 * align_up(sizeof(double) * (size_t)n_cols, 256) + align_up(sizeof(FusedPlan), 256) +
         align_up(sizeof(uint32_t) * (size_t)n_rows * K1, 256);
}

static FixedScales make_scales(float target_sum) {
  // 2^E > target_sum >= x' ;  2^EL > log1p(target_sum) >= x''
  int E = 0, EL = 0;
  frexp((double)target_sum, &E);                           // target_sum = m 2^E, m in [0.5, 1)
  frexp(log1p((double)target_sum) * 1.000001, &EL);
  if (E < 1) E = 1;
  if (EL < 1) EL = 1;
  FixedScales s;
  const int k1log = 52 - EL, k2log = 52 - 2 * EL, k1lin = 52 - E, k2hi = 52 - 2 * E,
            k2lo = 72 - 2 * E;
  s.m_s1log = (float)ldexp(1.0, k1log);
  s.m_s2log_h = (float)ldexp(1.0, k2log / 2);
  s.m_s1lin = (float)ldexp(1.0, k1lin);
  s.m_s2hi_h = (float)ldexp(1.0, k2hi / 2);
  s.m_s2lo_h = (float)ldexp(1.0, k2lo / 2);
  s.lin_theta = (float)ldexp(1.0, E - 10);
  s.inv_s1log = ldexp(1.0, -k1log);
  s.inv_s2log = ldexp(1.0, -k2log);
  s.inv_s1lin = ldexp(1.0, -k1lin);
  s.inv_s2hi = ldexp(1.0, -k2hi);
  s.inv_s2lo = ldexp(1.0, -k2lo);
  return s;
}

template <bool LOG, bool LIN, bool FIXED>
static int launch_stream(const FusedArgs& a, size_t smem, cudaStream_t st) {
  static bool attr_set = false;
  if (!attr_set) {
    RSC_CUDA(cudaFuncSetAttribute(fused_stream_kernel<LOG, LIN, FIXED>,
                                  cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem));
    attr_set = true;
  }
  fused_stream_kernel<LOG, LIN, FIXED><<<fused_grid(), kFuThreads, smem, st>>>(a);
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
  if (!fused_fast_ok(X, target_sum, which) || X.n_rows == 0) {
    rc = launch_fused_generic(X, target_sum, cell_total_i64, which, S1log, S2log, S1lin, S2lin, st);
    if (rc != RSC_OK) return rc;
  } else {
    const bool fixed = !(which & RSC_MOMENTS_FP64_ACC);
    if (which & RSC_MOMENTS_LOG) {
      RSC_CUDA(cudaMemsetAsync(S1log, 0, sizeof(double) * G, st));
      RSC_CUDA(cudaMemsetAsync(S2log, 0, sizeof(double) * G, st));
    }
    if (which & RSC_MOMENTS_LIN) {
      RSC_CUDA(cudaMemsetAsync(S1lin, 0, sizeof(double) * G, st));
      RSC_CUDA(cudaMemsetAsync(S2lin, 0, sizeof(double) * G, st));
    }
    FusedPlan* plan = reinterpret_cast<FusedPlan*>(w + 4 * gsz);
    if (row_splits == nullptr) {
      uint32_t* sp = reinterpret_cast<uint32_t*>(w + 4 * gsz + align_up(sizeof(FusedPlan), 256));
      if ((rc = launch_row_splits(X, sp, st)) != RSC_OK) return rc;
      row_splits = sp;
    }
    const int wpg = words_per_gene(which, fixed);
    FusedArgs a;
    a.n_rows = X.n_rows; a.n_cols = X.n_cols; a.n_fine = split_blocks(X.n_cols);
    a.fine_per_group = (int)((kMaxDynSmem - 64) / ((size_t)wpg * 4 * RSC_SPLIT_WIDTH));
    if (a.fine_per_group > a.n_fine) a.fine_per_group = a.n_fine;
    a.Gt = a.fine_per_group * RSC_SPLIT_WIDTH;
    a.indptr = X.indptr; a.indices = X.indices; a.data = X.data; a.cell_total = cell_total_i64;
    a.splits = row_splits; a.target_sum = target_sum; a.fs = make_scales(target_sum);
    a.row_budget = (uint32_t)g_opt.fused_row_budget;
    a.S1log = S1log; a.S2log = S2log; a.S1lin = S1lin; a.S2lin = S2lin; a.plan = plan;
    fused_plan_kernel<<<1, 1024, 0, st>>>(plan, X.n_cols, a.n_fine, a.fine_per_group, fused_grid(),
                                          gene_n_cells);
    RSC_LAUNCH_CHECK("fused_plan_kernel");
    const size_t smem = (size_t)wpg * 4 * (size_t)a.Gt;
    switch ((which & 3) | (fixed ? 4 : 0)) {
      case 1: rc = launch_stream<true, false, false>(a, smem, st); break;
      case 2: rc = launch_stream<false, true, false>(a, smem, st); break;
      case 3: rc = launch_stream<true, true, false>(a, smem, st); break;
      case 5: rc = launch_stream<true, false, true>(a, smem, st); break;
      case 6: rc = launch_stream<false, true, true>(a, smem, st); break;
      default: rc = launch_stream<true, true, true>(a, smem, st); break;
    }
    if (rc != RSC_OK) return rc;
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

}  // namespace rsc
