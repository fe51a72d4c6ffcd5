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
//     the global outputs directly.  Every 512 rows of the CTA one warp checks the table and
//     moves the genes whose count or total field is half full to the global outputs (one
//     atomic AND per gene, while the other warps keep adding); fewer than 1020 rows are added
//     between two checks of a gene (1020 * 511 < 2^19), so no field can overflow into its
//     neighbour.  Whatever is left goes out once, at the end;
//   * optionally the row split table consumed by the fused pass (fused.cu): for every row,
//     the number of entries with column < k * RSC_SPLIT_WIDTH, found by comparing the column
//     block of a lane's last entry with its neighbour's (rows must be sorted).
#include <type_traits>

#include "common.cuh"

namespace rsc {

#ifndef RSC_QC_THREADS
#define RSC_QC_THREADS 1024
#endif
constexpr int kQcThreads = RSC_QC_THREADS;
constexpr int kQcWarps = kQcThreads / 32;
#ifndef RSC_QC_RG
#define RSC_QC_RG 2
#endif
constexpr int kQcRowsPerGrab = RSC_QC_RG;
#ifndef RSC_QC_AHEAD
#define RSC_QC_AHEAD 4
#endif
constexpr int kQcAhead = RSC_QC_AHEAD;
#ifndef RSC_QC_LONGROW
#define RSC_QC_LONGROW 6144
#endif
constexpr int kQcLongRow = RSC_QC_LONGROW;       // entries: rows longer than this look one step less ahead
#ifndef RSC_QC_EVICT
#define RSC_QC_EVICT 0        // bit 0: demand loads carry L2 evict_first; bit 1: look-ahead prefetches carry evict_last
#endif                  // L2 look-ahead of a warp, in steps of 128 entries
constexpr uint32_t kQcMaxFast = 511u;        // largest count that takes the shared-memory path
static_assert(512 + 3 * kQcWarps * kQcRowsPerGrab + 64 <= 1020, "QC pass: too many rows in flight for the lazy flush");

struct QcArgs {
  int64_t n_rows;
  int64_t nnz;
  int32_t n_cols;
  int32_t n_fine;            // K = number of column blocks (split table has K + 1 entries per row)
  uint32_t check_shift;      // a warp checks the CTA's table every 2^check_shift rows
  uint32_t flush_all;        // 1: a check moves every gene to the global outputs (testing)
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
  int32_t n_need;            // > 0: only the split entries need[0..n_need) are written
  int32_t need[32];
  unsigned long long* row_counter;
};

__device__ __forceinline__ long long warp_sum_ll(long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// native shared atomic add on a 32-bit shared address, returning the previous word
__device__ __forceinline__ uint32_t qc_atoms_add(uint32_t saddr, uint32_t v) {
  uint32_t old;
  asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(saddr), "r"(v));
  return old;
}

// count | total of one packed word -> the global outputs
__device__ __forceinline__ void qc_word_to_global(int g, uint32_t w, int32_t* gene_n_cells,
                                                  unsigned long long* gene_total) {
  const uint32_t c = (w >> 20) & 0x7ffu, t = w & 0xfffffu;
  if (c != 0u && gene_n_cells != nullptr) atomicAdd(&gene_n_cells[g], (int)c);
  if (t != 0u && gene_total != nullptr) atomicAdd(&gene_total[g], (unsigned long long)t);
}
// Table check by one warp while the others keep adding: genes with a half-full field leave
// the table (atomic AND: the flag bit stays, the old word is what goes out).  Out of line:
// it runs once per 512 rows and must not cost the streaming loop registers.
__device__ __noinline__ void qc_check_table(uint32_t* qsm, int G, int lane, uint32_t flush_all,
                                            int32_t* gene_n_cells, unsigned long long* gene_total) {
  for (int g = lane; g < G; g += 32) {
    const uint32_t w = *reinterpret_cast<volatile uint32_t*>(qsm + g);
    if (flush_all || (w & 0x40000000u) != 0u || (w & 0x80000u) != 0u)
      qc_word_to_global(g, atomicAnd(qsm + g, 0x80000000u), gene_n_cells, gene_total);
  }
}

// NB > 0: the table's NB interior entries (need[1 .. NB]; need[0] = 0 and need[NB + 1] = K are
// the trivial ones) are counted while the row streams by, from the columns the lanes hold anyway:
// an interior step asks one vote "is my quad's last column below the bound?" (rows are sorted, so
// the lanes below form a prefix), an edge step counts entry by entry.  NB = 0 with SPLITS: binary
// searches in the row after it was streamed (any number of entries).
template <bool SPLITS, int NB>
__global__ void __launch_bounds__(kQcThreads, 1) qc_stream_kernel(const QcArgs a) {
  extern __shared__ __align__(16) uint32_t qsm[];      // [G] packed flag | count | total, + 1 spare
  const int G = a.n_cols;
  const int tid = threadIdx.x, lane = tid & 31;
  const int K = a.n_fine;
  uint32_t sbase = (uint32_t)__cvta_generic_to_shared(qsm);
  asm volatile("mov.u32 %0, %0;" : "+r"(sbase));       // keep it in a register
  __shared__ unsigned s_rows;
  __shared__ volatile unsigned s_chk;
  const uint64_t pol = l2_evict_first_policy();

  for (int g = tid; g <= G; g += kQcThreads)
    qsm[g] = (g < G && a.flags != nullptr && a.flags[g] != 0) ? 0x80000000u : 0u;

  // Row grabs: >= n_rows means the matrix is exhausted (only lane 0 holds the result; it is
  // broadcast when needed).  s_rows counts the rows this CTA has taken; the warp whose grab
  // crosses a multiple of 2^check_shift raises s_chk; the next warp to finish a grab takes it
  // and checks the table.
  auto grab_issue = [&]() -> long long {
    long long r = 0;
    if (lane == 0) {
      const unsigned c = atomicAdd(&s_rows, (unsigned)kQcRowsPerGrab);
      r = (long long)atomicAdd(a.row_counter, (unsigned long long)kQcRowsPerGrab);
      if (((c ^ (c + (unsigned)kQcRowsPerGrab)) >> a.check_shift) != 0u) s_chk = 1u;
    }
    return r;
  };
  auto to_global = [&](int g, uint32_t w) { qc_word_to_global(g, w, a.gene_n_cells, a.gene_total); };
  auto check_table = [&]() { qc_check_table(qsm, G, lane, a.flush_all, a.gene_n_cells, a.gene_total); };
  auto load_ptrs = [&](long long r0) -> int64_t {       // lanes 0..RG: indptr[r0 + lane]
    int64_t p = 0;
    if (lane <= kQcRowsPerGrab && r0 + lane <= a.n_rows) p = a.indptr[r0 + lane];
    return p;
  };
  // L2 prefetch of the 128 entries at p0 (both arrays): lanes 0..3 touch one 128-byte line each;
  // bounded look-ahead, so nothing is evicted before it is used
  auto l2_prefetch = [&](int64_t p0) {
    const int64_t p = p0 + lane * 32;
    if (lane < 4 && p < a.nnz) {
#if RSC_QC_EVICT & 2
      asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(a.indices + p));
      asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(a.data + p));
#else
      asm volatile("prefetch.global.L2 [%0];" ::"l"(a.indices + p));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(a.data + p));
#endif
    }
  };
  auto opaque = [](int v) -> int { asm volatile("mov.u32 %0, %0;" : "+r"(v)); return v; };
  // per-lane partial sums of the current row.  acc packs the fast path's two sums in one word,
  // exactly as the table does: bits 0..19 the lane's total, bits 20..31 its detected-entry count
  // (one add per entry).  A lane sees at most 57 840 / 32 = 1808 entries of a row (canonical CSR,
  // n_cols <= kQcMaxGenes) of at most 511 each: 1808 * 511 < 2^20, so the fields cannot mix.
  unsigned acc, m32;                                    // fast path (counts 1 .. 511)
  long long T64, M64;                                   // slow path (large / negative counts)

  // One quad of 4 consecutive entries.  EDGE: only entries e0 + k in [0, len) belong to the
  // row; the others add 0 to the spare word qsm[G].
  // Fast path: every valid value truncates to an integer in 1 .. 511 (one unsigned compare on
  // xi - 1 covers explicit zeros, fractions below 1, negatives and large counts): the word
  // count | total = xi + 2^20 goes to the table with one atomic and to acc with one add; the
  // flagged-subset sum is touched only when a returned word carries the flag bit (few genes).
  auto quad = [&](auto edge_tag, const int4 jv, const float4 xv, int e0, int len) {
    constexpr bool EDGE = decltype(edge_tag)::value;
    const int j[4] = {jv.x, jv.y, jv.z, jv.w};
    const float x[4] = {xv.x, xv.y, xv.z, xv.w};
    int xi[4];
    unsigned worst = 0u;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const bool valid = !EDGE || (unsigned)(e0 + k) < (unsigned)len;
      xi[k] = __float2int_rz(x[k]);
      const unsigned d = valid ? (unsigned)(xi[k] - 1) : 0u;
      worst = max(worst, d);
    }
    if (worst < kQcMaxFast) {                           // all valid xi in 1 .. 511
      uint32_t old[4], add[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const bool valid = !EDGE || (unsigned)(e0 + k) < (unsigned)len;
        add[k] = valid ? (uint32_t)xi[k] + 0x100000u : 0u;
        const uint32_t jj = valid ? (uint32_t)j[k] : (uint32_t)G;
        old[k] = qc_atoms_add(sbase + (jj << 2), add[k]);
        acc += add[k];
      }
#ifdef RSC_QC_FLAGBRANCH
      if ((int)(old[0] | old[1] | old[2] | old[3]) < 0)   // a flagged gene among the four (rare)
#endif
      {
#pragma unroll
        for (int k = 0; k < 4; ++k) m32 += (add[k] & 0xfffffu) & (uint32_t)((int)old[k] >> 31);
      }
    } else {                                            // rare: explicit zeros, fractions, counts > 511, negative, non-finite
#pragma unroll 1
      for (int k = 0; k < 4; ++k) {
        if (EDGE && !((unsigned)(e0 + k) < (unsigned)len)) continue;
        const float xv1 = k == 0 ? x[0] : k == 1 ? x[1] : k == 2 ? x[2] : x[3];
        const int jj = k == 0 ? j[0] : k == 1 ? j[1] : k == 2 ? j[2] : j[3];
        const int xi1 = __float2int_rz(xv1);
        const bool nz = xv1 != 0.0f;
        if ((unsigned)xi1 <= kQcMaxFast) {
          const uint32_t a1 = (uint32_t)xi1 + (nz ? 0x100000u : 0u);
          const uint32_t o = qc_atoms_add(sbase + ((uint32_t)jj << 2), a1);
          acc += a1;
          m32 += (uint32_t)xi1 & (uint32_t)((int)o >> 31);
        } else {
          const long long xl = (long long)xv1;
          acc += nz ? 0x100000u : 0u;
          T64 += xl;
          if (qsm[jj] >> 31) M64 += xl;
          if (a.gene_n_cells != nullptr && nz) atomicAdd(&a.gene_n_cells[jj], 1);
          if (xl != 0 && a.gene_total != nullptr)
            atomicAdd(&a.gene_total[jj], (unsigned long long)xl);
        }
      }
    }
  };

  {
    if (tid == 0) { s_rows = 0u; s_chk = 0u; }
    __syncthreads();
    // Grabs are pipelined two deep (see fused.cu): row range of grab g + 1 known and its
    // indptr entries loaded while grab g is processed; every row is prefetched into L2 one
    // row ahead of its use.
    long long r0 = __shfl_sync(0xffffffffu, grab_issue(), 0);
    int64_t mptr = r0 < a.n_rows ? load_ptrs(r0) : 0;
    long long rnext = __shfl_sync(0xffffffffu, grab_issue(), 0);
    while (r0 < a.n_rows) {
      const long long pending = grab_issue();
      const bool next_ok = rnext < a.n_rows;
      const int64_t nptr = next_ok ? load_ptrs(rnext) : 0;
      const int nr = (int)min((long long)kQcRowsPerGrab, a.n_rows - r0);
      const int64_t gend = __shfl_sync(0xffffffffu, mptr, nr);   // end of the grab's contiguous range
      // where the look-ahead continues once it runs past gend: the head of the next grab.  The
      // distance stays kQcAhead steps across the grab boundary -- fetching that head any earlier
      // (a whole row ahead) lets part of it fall out of L2 again before it is used
      const int64_t nhead = next_ok ? (__shfl_sync(0xffffffffu, nptr, 0) & ~3LL) : a.nnz;
#pragma unroll 1
      for (int ri = 0; ri < nr; ++ri) {
        const long long row = r0 + ri;
        const int64_t beg = __shfl_sync(0xffffffffu, mptr, ri);
        const int64_t end = __shfl_sync(0xffffffffu, mptr, ri + 1);
        // quads at 16-byte aligned offsets; e = index relative to the row start.  The lane's
        // pointers / e0 advance by 128 entries per step (no per-step address arithmetic).
        const int64_t abeg = beg & ~3LL;
        const int head = (int)(beg - abeg);
        const int len = (int)(end - beg);
        const int span = opaque(len > 0 ? head + len : 0);
        acc = 0; m32 = 0; T64 = 0; M64 = 0;
        unsigned n32x = 0u;                               // NB = 1: the edge-step split count rides on the n_genes sum
        int cnt_i[NB > 0 ? NB : 1], cnt_e[NB > 0 ? NB : 1];   // entries below bound b: interior steps (warp-uniform) / edge steps (per lane)
#pragma unroll
        for (int b = 0; b < NB; ++b) { cnt_i[b] = 0; cnt_e[b] = 0; }
        uint32_t* sp = SPLITS ? a.splits + (size_t)row * (size_t)(K + 1) : nullptr;
        const int32_t* ip = a.indices + abeg + lane * 4;
        const float* dp = a.data + abeg + lane * 4;
        int e0 = lane * 4 - head;
        // every quad of the row lies inside the arrays (false only for the matrix's last row)
        const bool vec_ok = opaque(abeg + ((span + 3) & ~3) <= a.nnz ? 1 : 0) != 0;
        auto load_q = [&](const int32_t* ipq, const float* dpq, int e, int4& jv, float4& xv) {
          if (e >= len) return;                         // quad past the row
          if (vec_ok) {
#if RSC_QC_EVICT & 1
            jv = ldg_stream_i4(ipq, pol);
            xv = ldg_stream_f4(dpq, pol);
#else
            jv = __ldg(reinterpret_cast<const int4*>(ipq));
            xv = __ldg(reinterpret_cast<const float4*>(dpq));
#endif
          } else {
            jv = make_int4(0, 0, 0, 0);
            xv = make_float4(0.f, 0.f, 0.f, 0.f);
            if (e + 0 < len) { jv.x = __ldg(ipq + 0); xv.x = __ldg(dpq + 0); }
            if (e + 1 < len) { jv.y = __ldg(ipq + 1); xv.y = __ldg(dpq + 1); }
            if (e + 2 < len) { jv.z = __ldg(ipq + 2); xv.z = __ldg(dpq + 2); }
            if (e + 3 < len) { jv.w = __ldg(ipq + 3); xv.w = __ldg(dpq + 3); }
          }
        };
        int4 jn = make_int4(0, 0, 0, 0);
        float4 xn = make_float4(0.f, 0.f, 0.f, 0.f);
        if (span > 0) load_q(ip, dp, e0, jn, xn);
        // L2 look-ahead position (lane-uniform): kQcAhead steps ahead, one step less inside long rows
        // (measured: 4 steps serve ordinary rows best, cfg3 1.84 vs 1.87 ms with 3; the very long rows of
        // cfg5's tail want 3: 1.97 vs 2.10 ms -- a longer distance costs DRAM re-reads there)
        int64_t pf = abeg + (len > kQcLongRow ? kQcAhead - 1 : kQcAhead) * 128;
#pragma unroll 2
        for (int base = 0; base < span; base += 128) {
          const int4 jc = jn;
          const float4 xc = xn;
          load_q(ip + 128, dp + 128, e0 + 128, jn, xn);
          l2_prefetch(pf < gend ? pf : nhead + ((pf - gend) & ~127LL));
          const bool inter = (base > 0 || head == 0) && (base + 128 <= span);
          if (inter) {
            quad(std::false_type{}, jc, xc, e0, len);
#pragma unroll
            for (int b = 0; b < NB; ++b) {
              if (cnt_i[b] >= 0) {                      // warp-uniform: the bound was not crossed yet
                const int32_t bound = a.need[b + 1] << RSC_SPLIT_SHIFT;
                const unsigned mge = __ballot_sync(0xffffffffu, jc.w >= bound);
                if (mge == 0u) {
                  cnt_i[b] += 128;
                } else {                                // the crossing step: count it, then stop looking
                  const int L = __ffs(mge) - 1;
                  const int part = (jc.x < bound ? 1 : 0) + (jc.y < bound ? 1 : 0) + (jc.z < bound ? 1 : 0);
                  cnt_i[b] = ~(cnt_i[b] + 4 * L + __shfl_sync(0xffffffffu, part, L));
                }
              }
            }
          } else if (e0 < len) {
            quad(std::true_type{}, jc, xc, e0, len);
#pragma unroll
            for (int b = 0; b < NB; ++b) {
              const int32_t bound = a.need[b + 1] << RSC_SPLIT_SHIFT;
              cnt_e[b] += ((unsigned)(e0 + 0) < (unsigned)len && jc.x < bound ? 1 : 0) +
                          ((unsigned)(e0 + 1) < (unsigned)len && jc.y < bound ? 1 : 0) +
                          ((unsigned)(e0 + 2) < (unsigned)len && jc.z < bound ? 1 : 0) +
                          ((unsigned)(e0 + 3) < (unsigned)len && jc.w < bound ? 1 : 0);
            }
          }
          ip += 128; dp += 128; e0 += 128; pf += 128;
        }
        if (SPLITS && NB > 0) {
          // cnt_i is stored complemented once the bound was crossed in an interior step.  NB = 1:
          // the edge-step count rides in the upper half of n32 (both < 2^16: n_cols < 57 841)
          if (NB == 1) n32x = (unsigned)cnt_e[0] << 16;
        } else if (SPLITS) {
          // split table of the row: lane k finds #{entries with column < k * RSC_SPLIT_WIDTH} by
          // binary search in the (sorted) row, whose lines were just streamed (L2 / L1 hits)
          // (all K + 1 entries, or only the listed ones: fewer probing lanes, less re-read traffic)
          const int nk = a.n_need > 0 ? a.n_need : K + 1;
          for (int i = lane; i < nk; i += 32) {
            const int k = a.n_need > 0 ? a.need[i] : i;
            const int32_t bound = k << RSC_SPLIT_SHIFT;
            int lo = 0, hi = len;
            if (k == 0) hi = 0;
            else if (k >= K) lo = len;
            while (lo < hi) {
              const int mid = (lo + hi) >> 1;
              if (__ldg(a.indices + beg + mid) < bound) lo = mid + 1; else hi = mid;
            }
            sp[k] = (uint32_t)lo;
          }
        }
        const unsigned t32 = acc & 0xfffffu;
        const unsigned n32 = (acc >> 20) + n32x;
        long long T, M;
        if (__any_sync(0xffffffffu, (T64 | M64) != 0)) {
          T = warp_sum_ll(T64 + (long long)t32);
          M = warp_sum_ll(M64 + (long long)m32);
        } else {                                        // 511 * len < 2^32: the 32-bit sums are exact
          T = (long long)warp_sum(t32);
          M = (long long)warp_sum(m32);
        }
        int N = (int)warp_sum(n32);
        if (SPLITS && NB > 0) {
          int lo[NB > 0 ? NB : 1];
#pragma unroll
          for (int b = 0; b < NB; ++b) {
            const int ci = cnt_i[b] < 0 ? ~cnt_i[b] : cnt_i[b];
            lo[b] = ci + (NB == 1 ? (N >> 16) : warp_sum(cnt_e[b]));
          }
          if (NB == 1) N &= 0xffff;
          // lanes 0 .. NB + 1 write one entry each
          uint32_t v = lane == 0 ? 0u : (uint32_t)len;
#pragma unroll
          for (int b = 0; b < NB; ++b) if (lane == b + 1) v = (uint32_t)lo[b];
          if (lane <= NB + 1) sp[a.need[lane]] = v;
        }
        if (lane == 0) {
          if (a.cell_total) a.cell_total[row] = T;
          if (a.cell_total_f32) a.cell_total_f32[row] = (float)T;
          if (a.cell_n_genes) a.cell_n_genes[row] = N;
          if (a.cell_flag_total) a.cell_flag_total[row] = M;
          if (a.cell_flag_pct) a.cell_flag_pct[row] = (float)(100.0 * (double)M / (double)T);
        }
      }
      r0 = rnext; mptr = nptr;
      rnext = __shfl_sync(0xffffffffu, pending, 0);
      if (s_chk != 0u) {
        unsigned t = 0u;
        if (lane == 0) t = atomicExch(const_cast<unsigned*>(&s_chk), 0u);
        if (__shfl_sync(0xffffffffu, t, 0) != 0u) check_table();
      }
    }
    __syncthreads();
    // the matrix is exhausted: what is left in the table goes to the global outputs
    for (int g = tid; g < G; g += kQcThreads) to_global(g, qsm[g]);
  }
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
              uint32_t* row_splits, const int32_t* need_blocks, int32_t n_need_blocks, void* ws,
              size_t, cudaStream_t st) {
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
  const size_t smem = sizeof(uint32_t) * ((size_t)X.n_cols + 1) + 16;   // + the spare word
  a.n_fine = split_blocks(X.n_cols);
  a.indptr = X.indptr; a.indices = X.indices; a.data = X.data; a.flags = gene_flags;
  a.cell_total = cell_total_i64; a.cell_total_f32 = cell_total_f32; a.cell_n_genes = cell_n_genes;
  a.cell_flag_total = cell_flag_total_i64; a.cell_flag_pct = cell_flag_pct;
  a.gene_n_cells = gene_n_cells;
  a.gene_total = reinterpret_cast<unsigned long long*>(gene_total_i64);
  a.splits = row_splits;
  a.n_need = 0;
  if (need_blocks != nullptr && n_need_blocks > 0 && n_need_blocks <= 32) {
    a.n_need = n_need_blocks;
    for (int i = 0; i < n_need_blocks; ++i) a.need[i] = need_blocks[i];
  }
  a.row_counter = static_cast<unsigned long long*>(ws);
  a.check_shift = 0u;                                           // largest power of two <= the option (<= 512)
  while (a.check_shift < 9u && (2u << a.check_shift) <= (uint32_t)g_opt.qc_row_budget) ++a.check_shift;
  a.flush_all = g_opt.flush_all ? 1u : 0u;
  int64_t blocks = (X.n_rows + kQcWarps * kQcRowsPerGrab - 1) / (kQcWarps * kQcRowsPerGrab);
  const int cap = g_opt.grid_ctas.load() > 0 ? g_opt.grid_ctas.load() : sm_count();
  if (blocks > cap) blocks = cap;
  // in-stream counting serves a list {0, k1 < .. < kNB, K} with 1 <= NB <= 3 interior entries
  int nb = 0;
  if (row_splits != nullptr && a.n_need >= 3 && a.n_need <= 5 && a.need[0] == 0 &&
      a.need[a.n_need - 1] == a.n_fine) {
    nb = a.n_need - 2;
    for (int i = 1; i < a.n_need; ++i)
      if (a.need[i] <= a.need[i - 1]) nb = 0;
  }
  void (*kern)(const QcArgs) = qc_stream_kernel<false, 0>;
  if (row_splits != nullptr) {
    kern = nb == 1 ? qc_stream_kernel<true, 1> : nb == 2 ? qc_stream_kernel<true, 2>
         : nb == 3 ? qc_stream_kernel<true, 3> : qc_stream_kernel<true, 0>;
  }
  // the attribute is per device: set on every launch (cheap), not cached per process
  RSC_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem));
  kern<<<(unsigned)blocks, kQcThreads, smem, st>>>(a);
  RSC_LAUNCH_CHECK("qc_stream_kernel");
  return RSC_OK;
}

}  // namespace rsc
