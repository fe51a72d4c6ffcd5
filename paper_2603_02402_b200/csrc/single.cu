// Single-pass chain: QC metrics + normalize_total + log1p + log-scale per-gene moments in ONE pass
// over the matrix (PAPER.md:L85 QC metrics, L91 normalisation / log1p / per-gene mean and
// variance; SURVEY.md section 8(d) "theoretical single pass (row kept on-chip, QC folded in)":
// 12 B / nnz of DRAM traffic instead of the 20 B / nnz of the QC pass followed by the fused pass).
//
// Why two kernels were needed: x' = x * s / T_i needs the whole row's total T_i before any entry
// of the row can be normalised, and the per-gene accumulators of 30 k genes (12 B of moment words
// + the QC count | total) do not fit one SM's shared memory, so a CTA can only serve a gene RANGE,
// i.e. a part of every row.  Here the two CTAs of a thread-block cluster serve the two halves of
// the gene axis and work on the SAME rows: warp w of CTA 0 and warp w of CTA 1 are partners.  For
// every row
//   A. each partner streams its half of the row once from DRAM (CTA 0 forward from the row's
//      start until the columns leave its range, CTA 1 backward from the row's end; rows are
//      sorted, so no split table and no search is needed) and does the QC work on it: partial
//      cell total / detected genes / flagged total, per-gene count | total into a packed
//      shared-memory table;
//   X. the partners exchange their partial sums through distributed shared memory (a 32-byte
//      mailbox per warp and row parity, written with st.async and counted on an mbarrier of the
//      receiver, which the receiver polls locally -- no fences); CTA 0 also hands over the next row
//      (it alone draws rows from the global cursor);
//   B. each partner walks its half again -- now an L2 hit, the lines were fetched a few
//      microseconds ago -- normalises, takes log1p, stores x'' and adds the exact-integer moment
//      words of fused.cu's three-word scheme.
// Nothing else waits: a partner never blocks before it has published what the other one needs
// (no cycle), the two CTAs of a cluster are co-scheduled by the hardware, and a bounded spin with
// an error flag replaces a hang should the protocol ever be violated.
//
// Shared memory per CTA (14 B / gene, 16 384 genes): moment words 3 x u32 per gene; QC table one
// 16-bit field per gene, two genes per u32 word:
//     bit 15      the gene's QC flag        bits 8..14  detected entries of this flush period
//     bits 0..7   sum of (count - 1) of this flush period ("excess"; total = entries + excess)
// Counts 1..4 take the table (one native shared atomic per entry, which also returns the flag);
// larger counts (1.4 % of the entries of config 3) go to the global outputs directly.  Every 16
// rows of the CTA one warp scans the table with 128-bit loads and moves the words with a
// half / quarter-full field out (atomic AND), so that a field cannot overflow into its neighbour: a
// field below its threshold (64 entries, excess 64) receives at most kSpRowsBetweenQcChecks = 64
// more rows before it is looked at again (64 + 63 <= 127, 3 * 64 + 63 <= 255).
//
// Serves sorted rows, 16-byte aligned arrays, n_cols <= 32 768, log-scale moments only; anything
// else takes the two-kernel chain (chain.cu decides).
#include <cooperative_groups.h>
#include <math.h>

#include <type_traits>

#include "common.cuh"
#include "fused_acc.cuh"

namespace cg = cooperative_groups;

namespace rsc {

#ifndef RSC_SP_THREADS
#define RSC_SP_THREADS 736
#endif
constexpr int kSpThreads = RSC_SP_THREADS;
constexpr int kSpWarps = kSpThreads / 32;
constexpr int kSpSlots = 16384;                 // genes per CTA (table capacity)
constexpr int kSpMaxGenes = 2 * kSpSlots;
constexpr int kSpBlock = 256;                   // the boundary between the two ranges is a multiple of this
constexpr uint32_t kSpMaxFast = 511u;           // largest count on the packed per-lane accumulators
constexpr int kSpTableCap = 4;                  // largest count that takes the shared QC table
#ifndef RSC_SP_AHEAD
#define RSC_SP_AHEAD 4
#endif
constexpr int kSpAhead = RSC_SP_AHEAD;          // L2 look-ahead of the first read, in steps of 128 entries
constexpr int kSpQcCheckShift = 4;              // QC table scan every 16 rows of the CTA
constexpr int kSpRowsBetweenQcChecks = 64;
static_assert((1 << kSpQcCheckShift) + kSpWarps + 24 <= kSpRowsBetweenQcChecks, "single pass: QC fields too small");
static_assert(63 + kSpRowsBetweenQcChecks <= 127 && 63 + (kSpTableCap - 1) * kSpRowsBetweenQcChecks <= 255,
              "single pass: QC field thresholds");
static_assert(kCheckRows + 2 * kSpWarps + 16 <= kMaxRowsBetweenChecks, "single pass: moment words");
constexpr int kSpSamples = 2048;                // rows the plan looks at
constexpr uint32_t kSpSpinLimit = 1u << 21;        // polls (>= 64 ns apart) before a warp gives up: > 0.1 s

// shared memory layout (bytes)
constexpr size_t kSpLogBytes = (size_t)(kSpSlots + 1) * kLogWords * 4;          // + the spare slot
constexpr size_t kSpQcOff = (kSpLogBytes + 15) / 16 * 16;
constexpr size_t kSpQcBytes = (size_t)(kSpSlots / 2 + 4) * 4;                   // + the spare word, 16-byte multiple
constexpr size_t kSpMailOff = kSpQcOff + kSpQcBytes;
constexpr int kSpMailStride = 80;                // per warp: two 32-byte messages + two mbarriers
constexpr size_t kSpMailBytes = ((size_t)kSpWarps * kSpMailStride + 15) / 16 * 16;
constexpr size_t kSpSmem = kSpMailOff + kSpMailBytes;
static_assert(kSpSmem <= kMaxDynSmem, "single pass: tables do not fit");
static_assert(kSpQcOff % 16 == 0 && kSpMailOff % 16 == 0, "alignment");

struct SingleArgs {
  int64_t n_rows;
  int64_t nnz;
  int32_t n_cols;
  float target_sum;
  uint32_t check_shift;       // moment words: a warp checks the CTA's table every 2^check_shift rows
  uint32_t flush_all;
  const int64_t* indptr;
  const int32_t* indices;
  float* data;
  const uint8_t* flags;
  int64_t* cell_total;
  float* cell_total_f32;
  int32_t* cell_n_genes;
  int64_t* cell_flag_total;
  float* cell_flag_pct;
  int32_t* gene_n_cells;
  unsigned long long* gene_total;
  double* S1log;
  double* S2log;
  unsigned long long* acc_log;
  FusedPlan* plan;            // sc_log, row_counter[0], need[1] = first gene of CTA 1's range
  unsigned int* col_hist;     // [n_cols / kSpBlock + 1] sampled entries per column block (plan)
  unsigned long long* big;    // [n_big][n_cols] counts above kSpTableCap: detected entries << 40 | total, one copy per
  int32_t n_big;              //   group of clusters (a hot gene's adds would serialise on ONE address otherwise)
  unsigned int* err;          // set when a partner did not answer (protocol violated)
};

// ---- distributed shared memory
__device__ __forceinline__ uint32_t sp_map_peer(uint32_t saddr, uint32_t peer) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(peer));
  return r;
}
// 16 bytes to the partner's shared memory, counted on the partner's mbarrier (async proxy)
__device__ __forceinline__ void sp_send16(uint32_t peer_addr, unsigned long long v0, unsigned long long v1,
                                          uint32_t peer_bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
               ::"r"(peer_addr), "l"(v0), "l"(v1), "r"(peer_bar) : "memory");
}
__device__ __forceinline__ void sp_bar_init(uint32_t bar) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void sp_bar_arm(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool sp_bar_try(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0u;
}
__device__ __forceinline__ unsigned long long sp_lds_u64(uint32_t a) {
  unsigned long long v;
  asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t sp_lds_u32(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
  return v;
}

// one 16-bit field -> the global outputs
__device__ __forceinline__ void sp_field_to_global(int g, uint32_t h, int32_t* gene_n_cells,
                                                   unsigned long long* gene_total) {
  const uint32_t c = (h >> 8) & 0x7fu, t = c + (h & 0xffu);
  if (c != 0u && gene_n_cells != nullptr) atomicAdd(&gene_n_cells[g], (int)c);
  if (t != 0u && gene_total != nullptr) atomicAdd(&gene_total[g], (unsigned long long)t);
}
// QC table scan by one warp while the others keep adding (out of line: runs every 16 rows)
__device__ __noinline__ void sp_check_qc(uint32_t* qsm, int g0, int n_genes, int lane, uint32_t flush_all,
                                         int32_t* gene_n_cells, unsigned long long* gene_total) {
  const int n_words = (n_genes + 1) >> 1;
  for (int w4 = lane * 4; w4 < n_words; w4 += 128) {
    uint4 v;
    asm volatile("ld.volatile.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "r"((uint32_t)__cvta_generic_to_shared(qsm + w4)));
    const uint32_t any = (v.x | v.y | v.z | v.w) & 0x40C040C0u;
    if (!flush_all && any == 0u) continue;
    const uint32_t ww[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (w4 + k < n_words && (flush_all ? (ww[k] & 0x7fff7fffu) != 0u : (ww[k] & 0x40C040C0u) != 0u)) {
        const uint32_t old = atomicAnd(qsm + w4 + k, 0x80008000u);
        const int g = g0 + 2 * (w4 + k);
        sp_field_to_global(g, old & 0xffffu, gene_n_cells, gene_total);
        if (2 * (w4 + k) + 1 < n_genes) sp_field_to_global(g + 1, old >> 16, gene_n_cells, gene_total);
      }
    }
  }
}

// ------------------------------------------------------------------ the streaming kernel
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kSpThreads, 1)
single_pass_kernel(const SingleArgs a) {
  extern __shared__ __align__(16) uint32_t ssm[];
  __shared__ unsigned s_rows;
  __shared__ volatile unsigned s_abort;
  cg::cluster_group cluster = cg::this_cluster();
  const uint32_t rank = cluster.block_rank();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = a.n_cols;
  const int bnd = a.plan->need[1];                       // CTA 0: genes [0, bnd), CTA 1: [bnd, G)
  const int g0 = rank ? bnd : 0;
  const int Gn = rank ? G - bnd : bnd;                   // genes of this CTA (<= kSpSlots)
  const float mult_log = a.plan->sc_log.mult;

  uint32_t sb = (uint32_t)__cvta_generic_to_shared(ssm);
  asm volatile("mov.u32 %0, %0;" : "+r"(sb));            // keep it in a register
  uint32_t* qsm = ssm + kSpQcOff / 4;
  const uint32_t qb = sb + (uint32_t)kSpQcOff;
  const uint32_t mail = sb + (uint32_t)kSpMailOff + (uint32_t)warp * (uint32_t)kSpMailStride;   // my two mailbox slots (+64: their mbarriers)
  const uint32_t peer_mail = sp_map_peer(mail, rank ^ 1u);

  AccCtx cx;
  cx.sb_log = sb; cx.sb_lin = sb; cx.mult_log = mult_log; cx.mult_lin = 1.0f; cx.g0 = g0;
  cx.last_slot = (uint32_t)(Gn > 0 ? Gn - 1 : 0);
  cx.S1log = a.S1log; cx.S2log = a.S2log; cx.S1lin = nullptr; cx.S2lin = nullptr;
  const uint32_t last_slot = cx.last_slot;
  unsigned long long* big_base = a.big + (size_t)((blockIdx.x >> 1) % (unsigned)a.n_big) * (size_t)G;

  for (int i = tid; i < (int)(kSpLogBytes / 4); i += kSpThreads) ssm[i] = 0u;
  for (int i = tid; i < (int)(kSpQcBytes / 4); i += kSpThreads) {
    uint32_t w = 0u;
    const int s = 2 * i;
    if (a.flags != nullptr) {
      if (s < Gn && a.flags[g0 + s] != 0) w |= 0x8000u;
      if (s + 1 < Gn && a.flags[g0 + s + 1] != 0) w |= 0x80000000u;
    }
    qsm[i] = w;
  }
  for (int i = tid; i < (int)(kSpMailBytes / 4); i += kSpThreads) ssm[kSpMailOff / 4 + i] = 0u;
  if (tid == 0) { s_rows = 0u; s_abort = 0u; }
  __syncthreads();
  if (lane == 0) {                                       // one mbarrier per message slot, armed for the first two messages
    sp_bar_init(mail + 64u); sp_bar_init(mail + 72u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    sp_bar_arm(mail + 64u, 32u); sp_bar_arm(mail + 72u, 32u);
  }
  __syncthreads();
  cluster.sync();                                        // both CTAs' mailboxes are ready

  // a gene's moment words leave the CTA as 64-bit adds to the global integer totals (fused.cu)
  auto to_global_log = [&](int g, uint32_t w0, uint32_t s0, uint32_t W) {
    unsigned long long* acc = a.acc_log + g;
    const size_t G64 = (size_t)G;
    const uint32_t hi = W & ((1u << kLogCarryBit) - 1u);
    atomicAdd(acc, ((unsigned long long)(W >> kLogCarryBit) << 32) | w0);
    if (s0) atomicAdd(acc + 2 * G64, (unsigned long long)s0);
    if (hi) atomicAdd(acc + 3 * G64, (unsigned long long)hi);
  };
  auto check_log = [&]() {
    for (int s = lane; s < Gn; s += 32) {
      uint32_t* w = ssm + (size_t)s * kLogWords;
      const uint32_t W = *reinterpret_cast<volatile uint32_t*>(w + 2);
      if (a.flush_all || (W & ((1u << kLogCarryBit) - 1u)) >= (1u << (kLogCarryBit - 1)) ||
          (W >> kLogCarryBit) >= kLogCarryHalf) {
        const uint32_t w0 = atomicExch(w, 0u), s0 = atomicExch(w + 1, 0u), Wx = atomicExch(w + 2, 0u);
        if (w0 | s0 | Wx) to_global_log(g0 + s, w0, s0, Wx);
      }
    }
  };

  // ---- exchange.  Message of sequence number q >= 1 lives in slot q & 1:
  //   +0 partial cell total (i64)   +8 partial flagged total (i64)   +16 next row (i64, from CTA 0)
  //   +24 partial detected genes (u32)
  // and is complete when the slot's mbarrier has counted its 32 bytes (phase parity (q >> 1) & 1).
  auto post = [&](uint32_t q, long long T, long long M, long long next_row, uint32_t N) {
    if (lane == 0) {
      const uint32_t p = peer_mail + (q & 1u) * 32u, bar = peer_mail + 64u + (q & 1u) * 8u;
      sp_send16(p, (unsigned long long)T, (unsigned long long)M, bar);
      sp_send16(p + 16, (unsigned long long)next_row, (unsigned long long)N, bar);
    }
  };
  auto receive = [&](uint32_t q, long long& T, long long& M, long long& next_row, uint32_t& N) {
    long long t = 0, m = 0, r = 0;
    uint32_t n = 0;
    if (lane == 0) {
      const uint32_t p = mail + (q & 1u) * 32u, bar = mail + 64u + (q & 1u) * 8u;
      uint32_t spins = 0;
      while (!sp_bar_try(bar, (q >> 1) & 1u)) {
        if (s_abort != 0u || ++spins > kSpSpinLimit) {     // never hang: give up, flag the run
          s_abort = 1u;
          atomicExch(a.err, 1u);
          break;
        }
        __nanosleep(64);                                   // a poll costs 11 issue slots: leave them to the other warps
      }
      t = (long long)sp_lds_u64(p);
      m = (long long)sp_lds_u64(p + 8);
      r = (long long)sp_lds_u64(p + 16);
      n = sp_lds_u32(p + 24);
      sp_bar_arm(bar, 32u);                                // for message q + 2
      if (s_abort != 0u) r = a.n_rows;                     // stop this warp
    }
    T = __shfl_sync(0xffffffffu, t, 0);
    M = __shfl_sync(0xffffffffu, m, 0);
    next_row = __shfl_sync(0xffffffffu, r, 0);
    N = __shfl_sync(0xffffffffu, n, 0);
  };

  // ---- per-lane partial sums of the first read (as in qc.cu)
  unsigned acc, m32;                                     // packed total | detected count; flagged total
  long long T64, M64;                                    // counts beyond 511, negative values
  int cnt_e;                                             // stored entries of my range seen in edge quads

  // First read of one quad: QC work on the entries that belong to the row (position) AND to my
  // gene range (column).  Returns true when an entry of the row lay outside my range (the half
  // ends in this step).
  auto quad_a = [&](auto edge_tag, const int4 jv, const float4 xv, int e0, int len) -> bool {
    constexpr bool EDGE = decltype(edge_tag)::value;
    const int j[4] = {jv.x, jv.y, jv.z, jv.w};
    const float x[4] = {xv.x, xv.y, xv.z, xv.w};
    int xi[4];
    bool valid[4];
    bool out_any = false;
    unsigned worst = 0u;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      valid[k] = true;
      if (EDGE) {
        const bool pos = (unsigned)(e0 + k) < (unsigned)len;
        const bool inr = (unsigned)(j[k] - g0) < (unsigned)Gn;
        valid[k] = pos && inr;
        out_any = out_any || (pos && !inr);
        cnt_e += valid[k] ? 1 : 0;
      }
      xi[k] = __float2int_rz(x[k]);
      const unsigned d = valid[k] ? (unsigned)(xi[k] - 1) : 0u;
      worst = max(worst, d);
    }
    if (worst < kSpMaxFast) {                              // all valid xi in 1 .. 511
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t addv = valid[k] ? (uint32_t)xi[k] + 0x100000u : 0u;
        const uint32_t slot = valid[k] ? min((uint32_t)(j[k] - g0), (uint32_t)kSpSlots) : (uint32_t)kSpSlots;
        const uint32_t sh = (slot & 1u) << 4;
        const bool big = xi[k] > kSpTableCap;
        const uint32_t a16 = (valid[k] && !big) ? ((uint32_t)(xi[k] - 1) + 0x100u) << sh : 0u;
        const uint32_t old = atoms_add(qb + ((slot >> 1) << 2), a16);
        acc += addv;
        m32 += (addv & 0xfffffu) & (uint32_t)((int)(old << (16u - sh)) >> 31);
        if (valid[k] && big)                               // beyond the table's fields: one 64-bit add, count << 40 | total
          atomicAdd(big_base + j[k], (1ull << 40) | (unsigned long long)xi[k]);
      }
    } else {                                               // rare: explicit zeros, fractions, counts > 511, negative, non-finite
#pragma unroll 1
      for (int k = 0; k < 4; ++k) {
        const bool vk = k == 0 ? valid[0] : k == 1 ? valid[1] : k == 2 ? valid[2] : valid[3];
        if (!vk) continue;
        const float xv1 = k == 0 ? x[0] : k == 1 ? x[1] : k == 2 ? x[2] : x[3];
        const int jj = k == 0 ? j[0] : k == 1 ? j[1] : k == 2 ? j[2] : j[3];
        const int xi1 = __float2int_rz(xv1);
        const bool nz = xv1 != 0.0f;
        const uint32_t slot = min((uint32_t)(jj - g0), (uint32_t)kSpSlots);
        const uint32_t sh = (slot & 1u) << 4;
        if (nz && xi1 >= 1 && xi1 <= kSpTableCap) {
          const uint32_t old = atoms_add(qb + ((slot >> 1) << 2), ((uint32_t)(xi1 - 1) + 0x100u) << sh);
          acc += (uint32_t)xi1 + 0x100000u;
          m32 += (uint32_t)xi1 & (uint32_t)((int)(old << (16u - sh)) >> 31);
        } else {
          const bool flagged = ((qsm[slot >> 1] >> (15u + sh)) & 1u) != 0u;
          const long long xl = (long long)xv1;
          if ((unsigned)xi1 <= kSpMaxFast) {
            acc += (uint32_t)xi1 + (nz ? 0x100000u : 0u);
            if (flagged) m32 += (uint32_t)xi1;
          } else {
            acc += nz ? 0x100000u : 0u;
            T64 += xl;
            if (flagged) M64 += xl;
          }
          if (a.gene_n_cells != nullptr && nz) atomicAdd(&a.gene_n_cells[jj], 1);
          if (xl != 0 && a.gene_total != nullptr) atomicAdd(&a.gene_total[jj], (unsigned long long)xl);
        }
      }
    }
    return out_any;
  };

  // Second read of one quad (fused.cu's log-scale quad): normalise, log1p, moment words.
  auto quad_b = [&](auto edge_tag, const int4 jv, const float4 xv, float scale, int e0, int len) -> float4 {
    constexpr bool EDGE = decltype(edge_tag)::value;
    const int j[4] = {jv.x, jv.y, jv.z, jv.w};
    const float x[4] = {xv.x, xv.y, xv.z, xv.w};
    float xl[4], tl[4];
    bool valid[4];
    bool ok = true;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      valid[k] = !EDGE || (unsigned)(e0 + k) < (unsigned)len;
      const float xn = __fmul_rn(x[k], scale);
      xl[k] = log1p_ge_quarter(xn);
      tl[k] = xl[k] * mult_log;
      ok = ok && (in_window_log(tl[k]) || !valid[k]);
    }
    if (ok) {
      uint32_t so3[4], al[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t slot = valid[k] ? min((uint32_t)(j[k] - g0), last_slot) : (uint32_t)kSpSlots;
        so3[k] = slot * (kLogWords * 4u);
        al[k] = valid[k] ? __float2uint_rz(tl[k]) : 0u;
      }
      acc3_quad(sb, so3, al);
    } else {
      const uint32_t vm = (valid[0] ? 1u : 0u) | (valid[1] ? 2u : 0u) | (valid[2] ? 4u : 0u) |
                          (valid[3] ? 8u : 0u);
      return quad_rare<true, false, false>(cx, jv, xv, scale, vm, (uint32_t)kSpSlots);
    }
    return make_float4(xl[0], xl[1], xl[2], xl[3]);
  };

  // ---- rows.  CTA 0 draws them from the global cursor, one grab ahead, and hands every row to
  // its partner with the message that precedes it (message 0 carries the first row).
  const int dstep = rank ? -1 : 1;
  auto grab_issue = [&]() -> long long {
    long long r = 0;
    if (lane == 0) r = (long long)atomicAdd(&a.plan->row_counter[0], 1ull);
    return r;
  };
  auto load_ptrs = [&](long long r) -> int64_t {          // lanes 0, 1: indptr[r + lane]
    int64_t p = 0;
    if (lane <= 1 && r + lane <= a.n_rows) p = a.indptr[r + lane];
    return p;
  };
  // the first kSpAhead steps of my half of a row go to L2 (CTA 0: the row's start; CTA 1: its end)
  auto prefetch_head = [&](int64_t beg, int64_t end) {
    const int64_t lo = beg & ~31LL;
    int64_t p;
    if (rank == 0) p = lo + lane * 32;
    else p = ((end - 1) & ~31LL) - lane * 32;
    if (lane < kSpAhead * 4 && p >= lo && p < end) {
      asm volatile("prefetch.global.L2 [%0];" ::"l"(a.indices + p));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(a.data + p));
    }
  };

  long long row, row_next = 0, pending = 0;
  uint32_t q = 0;                                          // messages exchanged so far
  if (rank == 0) {
    row = __shfl_sync(0xffffffffu, grab_issue(), 0);
    post(0u, 0, 0, row, 0u);
    row_next = __shfl_sync(0xffffffffu, grab_issue(), 0);
    pending = grab_issue();
    long long t, m, r;
    uint32_t n;
    receive(0u, t, m, r, n);                               // (empty: keeps the two directions in step)
  } else {
    long long t, m;
    uint32_t n;
    post(0u, 0, 0, 0, 0u);
    receive(0u, t, m, row, n);
  }
  int64_t mptr = row < a.n_rows ? load_ptrs(row) : 0;
  if (row < a.n_rows) {
    const int64_t b0 = __shfl_sync(0xffffffffu, mptr, 0), e0 = __shfl_sync(0xffffffffu, mptr, 1);
    prefetch_head(b0, e0);
  }

  while (row < a.n_rows) {
    ++q;
    const int64_t beg = __shfl_sync(0xffffffffu, mptr, 0);
    const int64_t end = __shfl_sync(0xffffffffu, mptr, 1);
    const int64_t abeg = beg & ~3LL;
    const int head = (int)(beg - abeg);
    const int len = (int)(end - beg);
    const int span = len > 0 ? head + len : 0;
    const int nst = (span + 127) >> 7;
    // every quad of the row lies inside the arrays (false only for the matrix's last row)
    const bool vec_ok = abeg + ((span + 3) & ~3) <= a.nnz;
    auto load_q = [&](int64_t off, int e, int4& jv, float4& xv) {
      if (e >= len || e + 3 < 0) return;                   // quad outside the row
      if (vec_ok) {
        jv = __ldg(reinterpret_cast<const int4*>(a.indices + off));
        xv = *reinterpret_cast<const float4*>(a.data + off);
      } else {
        jv = make_int4(0, 0, 0, 0);
        xv = make_float4(0.f, 0.f, 0.f, 0.f);
        if (e + 0 < len) { jv.x = __ldg(a.indices + off + 0); xv.x = a.data[off + 0]; }
        if (e + 1 < len) { jv.y = __ldg(a.indices + off + 1); xv.y = a.data[off + 1]; }
        if (e + 2 < len) { jv.z = __ldg(a.indices + off + 2); xv.z = a.data[off + 2]; }
        if (e + 3 < len) { jv.w = __ldg(a.indices + off + 3); xv.w = a.data[off + 3]; }
      }
    };

    // ---- A: first read of my half, QC sums
    acc = 0; m32 = 0; T64 = 0; M64 = 0; cnt_e = 0;
    int cnt_i = 0;                                         // entries of interior steps (warp-uniform)
    {
      int st = rank ? nst - 1 : 0;
      int4 jn = make_int4(0, 0, 0, 0);
      float4 xn = make_float4(0.f, 0.f, 0.f, 0.f);
      int64_t off = abeg + (int64_t)st * 128 + lane * 4;
      int e0 = st * 128 + lane * 4 - head;
      if (nst > 0) load_q(off, e0, jn, xn);
      bool more = nst > 0;
      while (more) {
        const int4 jc = jn;
        const float4 xc = xn;
        const int stn = st + dstep;
        const bool has_next = (unsigned)stn < (unsigned)nst;
        if (has_next) load_q(off + dstep * 128, e0 + dstep * 128, jn, xn);
        {                                                  // L2 look-ahead, kSpAhead steps further on
          const int sp = st + dstep * kSpAhead;
          const int64_t p = abeg + (int64_t)sp * 128 + lane * 32;
          if (lane < 4 && (unsigned)sp < (unsigned)nst && p < a.nnz) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.indices + p));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.data + p));
          }
        }
        const bool pos_inter = (st > 0 || head == 0) && (st * 128 + 128 <= span);
        bool stop;
        if (pos_inter) {
          const int far = rank ? jc.x : jc.w;              // the quad's column farthest into the other range
          const unsigned mout = __ballot_sync(0xffffffffu, (unsigned)(far - g0) >= (unsigned)Gn);
          if (mout == 0u) {
            quad_a(std::false_type{}, jc, xc, e0, len);
            cnt_i += 128;
            stop = false;
          } else {
            quad_a(std::true_type{}, jc, xc, e0, len);
            stop = true;
          }
        } else {
          const bool o = quad_a(std::true_type{}, jc, xc, e0, len);
          stop = __any_sync(0xffffffffu, o);
        }
        more = has_next && !stop;
        st = stn; off += dstep * 128; e0 += dstep * 128;
      }
    }
    long long T, M;
    {
      const unsigned t32 = acc & 0xfffffu;
      if (__any_sync(0xffffffffu, (T64 | M64) != 0)) {
        T = warp_sum(T64 + (long long)t32);
        M = warp_sum(M64 + (long long)m32);
      } else {                                             // 511 * len < 2^32: the 32-bit sums are exact
        T = (long long)warp_sum(t32);
        M = (long long)warp_sum(m32);
      }
    }
    // detected genes (low half) and edge-quad entries of my range (high half) in one warp sum
    const unsigned NN = warp_sum((acc >> 20) + ((unsigned)cnt_e << 16));
    const int n_mine = cnt_i + (int)(NN >> 16);
    uint32_t N = NN & 0xffffu;

    // ---- X: exchange the partial sums (and the next row)
    if (rank == 0) {
      post(q, T, M, row_next, N);
    } else {
      post(q, T, M, 0, N);
    }
    // my segment of the row for the second read
    const int64_t sbeg = rank ? end - n_mine : beg;
    {
      long long To, Mo, rn;
      uint32_t No;
      receive(q, To, Mo, rn, No);
      T += To; M += Mo; N += No;
      if (rank != 0) row_next = rn;
      if (s_abort != 0u) row_next = a.n_rows;              // a partner gave up: stop (the run is flagged)
    }
    if (rank == 0 && lane == 0) {
      if (a.cell_total) a.cell_total[row] = T;
      if (a.cell_total_f32) a.cell_total_f32[row] = (float)T;
      if (a.cell_n_genes) a.cell_n_genes[row] = (int)N;
      if (a.cell_flag_total) a.cell_flag_total[row] = M;
      if (a.cell_flag_pct) a.cell_flag_pct[row] = (float)(100.0 * (double)M / (double)T);
    }
    const float scale = cell_scale(a.target_sum, T);
    // the next row's pointers are requested now and used after the second read
    const bool next_ok = row_next < a.n_rows;
    const int64_t nptr = next_ok ? load_ptrs(row_next) : 0;

    // ---- B: second read of my segment (L2), normalise + log1p + moment words, x'' written back
    {
      const int64_t sab = sbeg & ~3LL;
      const int shead = (int)(sbeg - sab);
      const int slen = n_mine;
      const int nq = slen > 0 ? (shead + slen + 3) >> 2 : 0;
      const int nsteps = (nq + 31) >> 5;
      auto interior = [&](int st) -> bool { return (st > 0 || shead == 0) && (st * 128 + 128 <= shead + slen); };
      auto load_step = [&](int st, int4& jv, float4& xv) {
        const int qd = st * 32 + lane;
        const int64_t off = sab + 4 * qd;
        if (interior(st)) {
          jv = __ldg(reinterpret_cast<const int4*>(a.indices + off));
          xv = *reinterpret_cast<const float4*>(a.data + off);
        } else if (qd < nq) {
          if (off + 4 <= a.nnz) {
            jv = __ldg(reinterpret_cast<const int4*>(a.indices + off));
            xv = *reinterpret_cast<const float4*>(a.data + off);
          } else {                                         // the last quad of the whole matrix
            const int e = qd * 4 - shead;
            jv = make_int4(0, 0, 0, 0);
            xv = make_float4(0.f, 0.f, 0.f, 0.f);
            if (e + 0 < slen) { jv.x = __ldg(a.indices + off + 0); xv.x = a.data[off + 0]; }
            if (e + 1 < slen) { jv.y = __ldg(a.indices + off + 1); xv.y = a.data[off + 1]; }
            if (e + 2 < slen) { jv.z = __ldg(a.indices + off + 2); xv.z = a.data[off + 2]; }
          }
        }
      };
      int4 jn = make_int4(0, 0, 0, 0);
      float4 xn4 = make_float4(0.f, 0.f, 0.f, 0.f);
      if (nsteps > 0) load_step(0, jn, xn4);
#pragma unroll 1
      for (int st = 0; st < nsteps; ++st) {
        const int4 jc = jn;
        const float4 xc = xn4;
        if (st + 1 < nsteps) load_step(st + 1, jn, xn4);
        const int qd = st * 32 + lane;
        const int e = qd * 4 - shead;
        float* dq = a.data + (sab + 4 * qd);
        if (interior(st)) {
          const float4 r = quad_b(std::false_type{}, jc, xc, scale, e, slen);
          st_once(reinterpret_cast<float4*>(dq), r);
        } else if (qd < nq) {
          const float4 r = quad_b(std::true_type{}, jc, xc, scale, e, slen);
          if (e >= 0 && e + 4 <= slen) {
            *reinterpret_cast<float4*>(dq) = r;
          } else {
            if ((unsigned)(e + 0) < (unsigned)slen) dq[0] = r.x;
            if ((unsigned)(e + 1) < (unsigned)slen) dq[1] = r.y;
            if ((unsigned)(e + 2) < (unsigned)slen) dq[2] = r.z;
            if ((unsigned)(e + 3) < (unsigned)slen) dq[3] = r.w;
          }
        }
        if (st == 0 && next_ok) {                          // the next row's head goes to L2 meanwhile
          const int64_t nb = __shfl_sync(0xffffffffu, nptr, 0), ne = __shfl_sync(0xffffffffu, nptr, 1);
          prefetch_head(nb, ne);
        }
      }
      if (nsteps == 0 && next_ok) {
        const int64_t nb = __shfl_sync(0xffffffffu, nptr, 0), ne = __shfl_sync(0xffffffffu, nptr, 1);
        prefetch_head(nb, ne);
      }
    }

    // ---- next row; table checks by the warp whose row crosses a check point
    row = row_next;
    mptr = nptr;
    if (rank == 0) {
      row_next = __shfl_sync(0xffffffffu, pending, 0);
      pending = grab_issue();
    }
    unsigned c = 0u;
    if (lane == 0) c = atomicAdd(&s_rows, 1u);
    c = __shfl_sync(0xffffffffu, c, 0);
    if (((c ^ (c + 1u)) >> kSpQcCheckShift) != 0u)
      sp_check_qc(qsm, g0, Gn, lane, a.flush_all, a.gene_n_cells, a.gene_total);
    if (((c ^ (c + 1u)) >> a.check_shift) != 0u) check_log();
  }

  __syncthreads();
  // the matrix is exhausted: everything left in the tables goes to the global outputs
  for (int s = tid; s < Gn; s += kSpThreads) {
    const uint32_t* w = ssm + (size_t)s * kLogWords;
    if (w[0] | w[1] | w[2]) to_global_log(g0 + s, w[0], w[1], w[2]);
    const uint32_t h = (qsm[s >> 1] >> ((s & 1) << 4)) & 0x7fffu;
    if (h) sp_field_to_global(g0 + s, h, a.gene_n_cells, a.gene_total);
  }
  cluster.sync();                                          // nobody leaves while a partner may still write here
}

// ------------------------------------------------------------------ plan
// The windows of the moment words and the boundary between the two gene ranges are placed from a
// sample of kSpSamples rows spread evenly over the matrix: the sampled cells' totals give the
// binades of their smallest x'' (fused.cu places the log-scale window from the same histogram of
// ALL cells; a value outside the window still lands in the global double sums -- correct, only
// slower), the sampled columns give the entries per block of kSpBlock genes.
__global__ void __launch_bounds__(256)
single_sample_kernel(SingleArgs a, int n_samples) {
  // the column histogram is collected per CTA in shared memory first: 3 M adds onto ~120 global addresses
  // took 0.8 ms
  __shared__ unsigned int hist[kSpMaxGenes / kSpBlock + 1];
  const int n_hist = a.n_cols / kSpBlock + 1;
  for (int i = threadIdx.x; i < n_hist; i += blockDim.x) hist[i] = 0u;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int wid = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int n_warps = (int)((gridDim.x * blockDim.x) >> 5);
  for (int sidx = wid; sidx < n_samples; sidx += n_warps) {
    const int64_t row = (int64_t)(((__int128)sidx * a.n_rows) / n_samples);
    const int64_t beg = a.indptr[row], end = a.indptr[row + 1];
    long long t = 0;
    for (int64_t p = beg + lane; p < end; p += 32) {
      t += (long long)a.data[p];
      atomicAdd(&hist[min(max(a.indices[p], 0), a.n_cols - 1) / kSpBlock], 1u);
    }
    t = warp_sum(t);
    if (lane == 0 && t > 0) {
      int e;
      frexpf(log1pf(__fdiv_rn(a.target_sum, (float)t)), &e);
      atomicAdd(&a.plan->depth_hist[min(max(e - 1 + 32, 0), 63)], 1u);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < n_hist; i += blockDim.x)
    if (hist[i]) atomicAdd(&a.col_hist[i], hist[i]);
}

__global__ void single_plan_kernel(SingleArgs a, int n_samples) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  FusedPlan* plan = a.plan;
  const double ts = (double)a.target_sum;
  {
    // log-scale window, as in fused_plan_kernel: bottom = binade of the smallest x'' of the sampled
    // cells (the deepest 1 / 1024 of them ignored), never above the top 2^E > log1p(target_sum),
    // never below 2^-2
    int E;
    frexp(log1p(ts) * 1.000001, &E);
    int L = E - kLogBinades;
    const unsigned long long skip = (unsigned long long)n_samples / 1024ull;
    unsigned long long below = 0ull;
    for (int b = 0; b < 64; ++b) {
      below += plan->depth_hist[b];
      if (below > skip) { L = min(b - 32, E - kLogBinades); break; }
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
  {
    // boundary: the block edge that halves the sampled entries, inside what the tables allow
    const int G = a.n_cols;
    const int nb = (G + kSpBlock - 1) / kSpBlock;
    unsigned long long total = 0ull;
    for (int b = 0; b < nb; ++b) total += a.col_hist[b];
    const int lo = max(1, (G - kSpSlots + kSpBlock - 1) / kSpBlock);    // G - bnd <= kSpSlots
    const int hi = min(nb - 1, kSpSlots / kSpBlock);                    // bnd <= kSpSlots
    int best = hi;
    unsigned long long cum = 0ull;
    for (int b = 0; b <= hi; ++b) {                                     // cum = sampled entries below block edge b
      if (b >= lo && 2ull * cum >= total) { best = b; break; }
      if (b < nb) cum += a.col_hist[b];
    }
    plan->need[0] = 0;
    plan->need[1] = min(best * kSpBlock, G);
    plan->need[2] = G;
    plan->n_groups = 2;
    plan->row_counter[0] = 0ull;
  }
}

// the copies of the large-count sums -> the per-gene outputs (after the streaming kernel)
__global__ void single_big_reduce_kernel(const unsigned long long* __restrict__ big, int n_big, int G,
                                         int32_t* __restrict__ gene_n_cells, unsigned long long* __restrict__ gene_total) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= G) return;
  unsigned long long c = 0ull, t = 0ull;
  for (int r = 0; r < n_big; ++r) {
    const unsigned long long v = big[(size_t)r * G + g];
    c += v >> 40;
    t += v & ((1ull << 40) - 1ull);
  }
  if (gene_n_cells != nullptr && c != 0ull) gene_n_cells[g] += (int32_t)c;
  if (gene_total != nullptr && t != 0ull) gene_total[g] += t;
}

// the run was flagged (a partner did not answer): poison the moments so that nobody trusts them
__global__ void single_guard_kernel(const unsigned int* err, int G, double* mean, double* var) {
  if (*err == 0u) return;
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g < G) {
    const double nan = __longlong_as_double(0x7ff8000000000000ll);
    if (mean) mean[g] = nan;
    if (var) var[g] = nan;
  }
}

// ------------------------------------------------------------------ host side
bool single_pass_ok(const rsc_csr& X, int which) {
  if (!(X.flags & RSC_CSR_SORTED) || g_opt.force_generic || !g_opt.single_pass) return false;
  if ((which & 7) != RSC_MOMENTS_LOG) return false;
  if (X.n_rows <= 0 || X.nnz <= 0 || X.n_cols < 2 * kSpBlock || X.n_cols > kSpMaxGenes) return false;
  if (X.n_rows >= (1LL << 24)) return false;              // 24-bit entry counts in the large-count sums
  if ((reinterpret_cast<uintptr_t>(X.indices) | reinterpret_cast<uintptr_t>(X.data)) & 15) return false;
  return true;
}

// copies of the large-count sums: one per 8192 rows, at most 32
static int single_n_big(int64_t n_rows) {
  const int64_t r = n_rows / 8192;
  return (int)(r < 1 ? 1 : r > 32 ? 32 : r);
}

size_t single_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t) {
  const size_t G = (size_t)n_cols;
  return align_up(sizeof(unsigned long long) * G * (size_t)single_n_big(n_rows), 256) + 2 * align_up(sizeof(double) * G, 256) + align_up(5 * sizeof(unsigned long long) * G, 256) +
         align_up(sizeof(FusedPlan), 256) + align_up(sizeof(unsigned int) * (G / kSpBlock + 2), 256) + 256;
}

int launch_single_pass(const rsc_csr& X, const uint8_t* gene_flags, float target_sum, int ddof,
                       int64_t* cell_total_i64, float* cell_total_f32, int32_t* cell_n_genes,
                       int64_t* cell_flag_total_i64, float* cell_flag_pct, int32_t* gene_n_cells,
                       int64_t* gene_total_i64, double* mean_log, double* var_log, void* ws, cudaStream_t st) {
  const size_t G = (size_t)X.n_cols;
  const size_t gsz = align_up(sizeof(double) * G, 256);
  const size_t asz = align_up(5 * sizeof(unsigned long long) * G, 256);
  const size_t psz = align_up(sizeof(FusedPlan), 256);
  const size_t hsz = align_up(sizeof(unsigned int) * (G / kSpBlock + 2), 256);
  unsigned char* w = static_cast<unsigned char*>(ws);
  const int n_big = single_n_big(X.n_rows);
  const size_t bsz = align_up(sizeof(unsigned long long) * G * (size_t)n_big, 256);
  RSC_CUDA(cudaMemsetAsync(w, 0, 2 * gsz + asz + psz + hsz + 256 + bsz, st));
  if (gene_n_cells) RSC_CUDA(cudaMemsetAsync(gene_n_cells, 0, sizeof(int32_t) * G, st));
  if (gene_total_i64) RSC_CUDA(cudaMemsetAsync(gene_total_i64, 0, sizeof(int64_t) * G, st));
  SingleArgs a;
  a.n_rows = X.n_rows; a.nnz = X.nnz; a.n_cols = X.n_cols; a.target_sum = target_sum;
  a.check_shift = 0u;
  while ((2u << a.check_shift) <= (uint32_t)kCheckRows && (2u << a.check_shift) <= (uint32_t)g_opt.fused_row_budget)
    ++a.check_shift;
  a.flush_all = g_opt.flush_all ? 1u : 0u;
  a.indptr = X.indptr; a.indices = X.indices; a.data = X.data; a.flags = gene_flags;
  a.cell_total = cell_total_i64; a.cell_total_f32 = cell_total_f32; a.cell_n_genes = cell_n_genes;
  a.cell_flag_total = cell_flag_total_i64; a.cell_flag_pct = cell_flag_pct;
  a.gene_n_cells = gene_n_cells;
  a.gene_total = reinterpret_cast<unsigned long long*>(gene_total_i64);
  a.S1log = reinterpret_cast<double*>(w);
  a.S2log = reinterpret_cast<double*>(w + gsz);
  a.acc_log = reinterpret_cast<unsigned long long*>(w + 2 * gsz);
  a.plan = reinterpret_cast<FusedPlan*>(w + 2 * gsz + asz);
  a.col_hist = reinterpret_cast<unsigned int*>(w + 2 * gsz + asz + psz);
  a.err = reinterpret_cast<unsigned int*>(w + 2 * gsz + asz + psz + hsz);
  a.big = reinterpret_cast<unsigned long long*>(w + 2 * gsz + asz + psz + hsz + 256);
  a.n_big = n_big;

  const int n_samples = (int)(X.n_rows < kSpSamples ? X.n_rows : kSpSamples);
  single_sample_kernel<<<(n_samples + 7) / 8, 256, 0, st>>>(a, n_samples);
  RSC_LAUNCH_CHECK("single_sample_kernel");
  single_plan_kernel<<<1, 32, 0, st>>>(a, n_samples);
  RSC_LAUNCH_CHECK("single_plan_kernel");

  int ctas = g_opt.grid_ctas.load() > 0 ? g_opt.grid_ctas.load() : sm_count();
  ctas &= ~1;
  if (ctas < 2) ctas = 2;
  RSC_CUDA(cudaFuncSetAttribute(single_pass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem));
  single_pass_kernel<<<ctas, kSpThreads, kSpSmem, st>>>(a);
  RSC_LAUNCH_CHECK("single_pass_kernel");
  single_big_reduce_kernel<<<(unsigned)((G + 255) / 256), 256, 0, st>>>(a.big, n_big, X.n_cols, gene_n_cells, a.gene_total);
  RSC_LAUNCH_CHECK("single_big_reduce_kernel");
  int rc = launch_fused_finish(X.n_cols, X.n_rows, ddof, a.plan, 0, a.acc_log, a.S1log, a.S2log, mean_log, var_log, st);
  if (rc != RSC_OK) return rc;
  single_guard_kernel<<<(unsigned)((G + 255) / 256), 256, 0, st>>>(a.err, X.n_cols, mean_log, var_log);
  RSC_LAUNCH_CHECK("single_guard_kernel");
  return RSC_OK;
}

}  // namespace rsc
