// Accumulator scheme of the streaming moment kernels (fused.cu, single.cu): constants, the plan
// kept in the workspace, and the exact-integer shared-memory accumulator primitives.  See the
// header of fused.cu for the design.
#pragma once

#include <math.h>

#include "common.cuh"

namespace rsc {


#ifndef RSC_FU_THREADS
#define RSC_FU_THREADS 736
#endif
constexpr int kFuThreads = RSC_FU_THREADS;
#ifndef RSC_FU_RG
#define RSC_FU_RG 2
#endif
constexpr int kFuRowsPerGrab = RSC_FU_RG;
#ifndef RSC_FU_HEAD
#define RSC_FU_HEAD 512
#endif
#ifndef RSC_FU_DIST
#define RSC_FU_DIST RSC_FU_HEAD
#endif
constexpr int kFuDist = RSC_FU_DIST;          // in-segment look-ahead distance, entries (<= kFuHead)
constexpr int kFuHead = RSC_FU_HEAD;              // entries of a segment requested from L2 before the segment is walked
constexpr long long kCheckBit = 1LL << 62;  // set in a grab's result: this grab crossed a check point
constexpr int kMaxGroups = 64;
// rows a CTA can add between two checks of a gene: the check interval (<= 512) + the grabs its
// warps hold (current, next, pending) must stay below kMaxRowsBetweenChecks (see check_tables)
#ifndef RSC_FU_CHECK
#define RSC_FU_CHECK 256
#endif
constexpr int kCheckRows = RSC_FU_CHECK;   // default / largest check interval (a power of two)
constexpr int kMaxRowsBetweenChecks = 410;
static_assert(kCheckRows + 3 * (kFuThreads / 32) * kFuRowsPerGrab + 16 <= kMaxRowsBetweenChecks,
              "fused pass: too many rows in flight for the lazy flush");
constexpr int kSetWords = 5;               // u32 words per gene of the linear-scale set (w0 w1 s0 s1 s2)
constexpr int kLogWords = 3;               // u32 words per gene of the log-scale set (w0 s0 W)
constexpr int kLogShift = 8;               // log-scale set: S2 accumulates (a * a + 2^7) >> 8
constexpr int kLogBinades = 5;             // log-scale set: 2^23 <= a < 2^28
constexpr int kLogCarryBit = 26;           // W = upper S2 word (bits 0..25) | carries of w0 (bits 26..31)
constexpr uint32_t kLogCarryHalf = 32u;    // half of the 6-bit carry field
// A gene is moved out when a field of W is half full, and a CTA adds at most
// kMaxRowsBetweenChecks = 410 rows between two checks of a gene:
//   upper S2 word: (a*a >> 8) >> 32 < 2^16 per add (+ carry), 410 * 2^16 < 2^25 = half of 26 bits;
//   carries of w0: at most 410 * 2^28 / 2^32 + 1 = 27 < 32 = half of 6 bits.
constexpr double kRowCost = 200.0;         // per-row-segment overhead, in entries (plan kernel)
constexpr int kMaxRangeBits = 19;          // 2^k * v_max <= 2^(23 + 19) = 2^42

struct MomentScale {                       // one per moment set; written by fused_plan_kernel
  float mult;                              // 2^k
  float pad;
  double inv1;                             // 2^-k
  double inv2;                             // 2^-2k
};

struct FusedPlan {                         // in the workspace
  int32_t n_groups;
  int32_t pad;
  int32_t cta_first[kMaxGroups + 1];
  unsigned long long row_counter[kMaxGroups];
  unsigned long long tmax;                 // largest cell total (fused_tmax_kernel)
  unsigned int depth_hist[64];             // cells by binade of log1p(target_sum / T_i), bin = exponent + 32
  MomentScale sc_log, sc_lin;
  // moments-only pass (rsc_gene_moments): chosen on the device by moments_plan_kernel
  int32_t scheme;                          // 1: three-word (narrow window) set, 2: five-word set
  int32_t Gt;                              // accumulator slots per CTA
  int32_t n_need;                          // n_groups + 1
  int32_t need[kMaxGroups + 1];            // column-block index at which group c starts
};
constexpr int kNeedStride = 8;             // split entries per row of the moments-only pass (<= 7 groups)

struct FusedArgs {
  int64_t n_rows;
  int32_t n_cols;
  int32_t n_fine;            // K
  int32_t fine_per_group;
  int32_t Gt;                // accumulator slots per CTA = fine_per_group * RSC_SPLIT_WIDTH
  int64_t nnz;
  const int64_t* indptr;
  const int32_t* indices;
  float* data;
  const int64_t* cell_total;
  const uint32_t* splits;   // fused: [n_rows][K + 1]; moments-only: [n_rows][kNeedStride], entry c = start of group c
  float target_sum;
  uint32_t row_budget;       // fp64 kernel: a CTA stops grabbing rows once it has taken this many (then flushes)
  uint32_t check_shift;      // integer kernels: a warp checks the CTA's tables every 2^check_shift rows
  uint32_t flush_all;        // 1: a check moves every gene to the global totals (testing)
  double* S1log; double* S2log; double* S1lin; double* S2lin;
  unsigned long long* acc_log;   // [5][n_cols] global totals of the words w0 w1 s0 s1 s2
  unsigned long long* acc_lin;
  FusedPlan* plan;
};

// ------------------------------------------------------------------ accumulator primitives
// native 32-bit shared atomics on 32-bit shared addresses
__device__ __forceinline__ uint32_t atoms_add(uint32_t saddr, uint32_t v) {
  uint32_t old;
  asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(saddr), "r"(v));
  return old;
}
__device__ __forceinline__ void reds_add(uint32_t saddr, uint32_t v) {
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(saddr), "r"(v));
}

// 2^23 <= t < 2^32 (t = v * 2^k): the float is an exact integer that fits one word
__device__ __forceinline__ bool in_window(float t) {
  return (__float_as_uint(t) - 0x4B000000u) < 0x04800000u;
}

// S1 += a, S2 += a * a for a one-word a; sa = shared byte address of the slot's word 0.
// Three returning atomics (w0, s0, s1) and two predicated carry increments (w1, s2).
__device__ __forceinline__ void acc_word(uint32_t sa, uint32_t a) {
  const unsigned long long q = (unsigned long long)a * a;
  const uint32_t q0 = (uint32_t)q, q1 = (uint32_t)(q >> 32);      // q1 <= 2^32 - 2
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      ".reg .u32 o, t;\n\t"
      "atom.shared.add.u32 o, [%0], %1;\n\t"
      "add.u32 t, o, %1;\n\t"
      "setp.lt.u32 p, t, o;\n\t"
      "@p red.shared.add.u32 [%0+4], 1;\n\t"
      "atom.shared.add.u32 o, [%0+8], %2;\n\t"
      "add.u32 t, o, %2;\n\t"
      "setp.lt.u32 p, t, o;\n\t"
      "selp.u32 t, 1, 0, p;\n\t"
      "add.u32 t, t, %3;\n\t"
      "atom.shared.add.u32 o, [%0+12], t;\n\t"
      "add.u32 o, o, t;\n\t"
      "setp.lt.u32 p, o, t;\n\t"
      "@p red.shared.add.u32 [%0+16], 1;\n\t"
      "}"
      ::"r"(sa), "r"(a), "r"(q0), "r"(q1));
}

// predicated carry increment of a shared word
__device__ __forceinline__ void reds_inc_if(uint32_t saddr, bool on) {
  if (on) asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(saddr));
}

// carry-out (0 / 1) of o + v
__device__ __forceinline__ uint32_t carry_of(uint32_t o, uint32_t v) {
  uint32_t c;
  asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, 0, 0;\n\t}" : "=r"(c) : "r"(o), "r"(v));
  return c;
}
// w + carry-out of (o + v)
__device__ __forceinline__ uint32_t add_carry_of(uint32_t w, uint32_t o, uint32_t v) {
  uint32_t r;
  asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %3, 0;\n\t}"
      : "=r"(r) : "r"(o), "r"(v), "r"(w));
  return r;
}

// acc_word for the 4 entries of a quad, staged so that the returning atomics of the four
// entries are in flight together (their slots are distinct: one row, four columns)
__device__ __forceinline__ void acc_quad(uint32_t base, const uint32_t (&so)[4], const uint32_t (&a)[4]) {
  uint32_t sa[4], o[4], o0[4], q0[4], q1[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) { sa[k] = base + so[k]; o[k] = atoms_add(sa[k], a[k]); }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    unsigned long long q;
    asm("mul.wide.u32 %0, %1, %1;" : "=l"(q) : "r"(a[k]));
    q0[k] = (uint32_t)q; q1[k] = (uint32_t)(q >> 32);             // q1 <= 2^32 - 2
    o0[k] = atoms_add(sa[k] + 8, q0[k]);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) reds_inc_if(sa[k] + 4, carry_of(o[k], a[k]) != 0u);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    q1[k] = add_carry_of(q1[k], o0[k], q0[k]);
    o[k] = atoms_add(sa[k] + 12, q1[k]);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) reds_inc_if(sa[k] + 16, carry_of(o[k], q1[k]) != 0u);
}

// ---- log-scale set: three words (w0 | s0 | W), branch-free
// 2^23 <= t < 2^29
__device__ __forceinline__ bool in_window_log(float t) {
  return (__float_as_uint(t) - 0x4B000000u) < (uint32_t)kLogBinades * 0x00800000u;
}
// W increment: upper word of b + carry-out of (o0 + b0) + (carry-out of (o + a) << kLogCarryBit)
__device__ __forceinline__ uint32_t log_top_word(uint32_t b1, uint32_t o0, uint32_t b0, uint32_t o, uint32_t a) {
  return add_carry_of(b1, o0, b0) + (carry_of(o, a) << kLogCarryBit);
}
__device__ __forceinline__ void acc3_word(uint32_t sa, uint32_t a) {
  unsigned long long q;
  asm("mad.wide.u32 %0, %1, %1, %2;" : "=l"(q) : "r"(a), "l"(1ull << (kLogShift - 1)));
  const uint32_t b0 = (uint32_t)(q >> kLogShift), b1 = (uint32_t)(q >> (32 + kLogShift));
  const uint32_t o = atoms_add(sa, a);
  const uint32_t o0 = atoms_add(sa + 4, b0);
  reds_add(sa + 8, log_top_word(b1, o0, b0, o, a));
}
// the 4 entries of a quad, staged so that the returning atomics are in flight together; an
// entry with a = 0 (masked) adds 0 to every word
__device__ __forceinline__ void acc3_quad(uint32_t base, const uint32_t (&so)[4], const uint32_t (&a)[4]) {
  uint32_t sa[4], o[4], o0[4], b0[4], b1[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) { sa[k] = base + so[k]; o[k] = atoms_add(sa[k], a[k]); }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    unsigned long long q;
    asm("mad.wide.u32 %0, %1, %1, %2;" : "=l"(q) : "r"(a[k]), "l"(1ull << (kLogShift - 1)));
    b0[k] = (uint32_t)(q >> kLogShift); b1[k] = (uint32_t)(q >> (32 + kLogShift));
    o0[k] = atoms_add(sa[k] + 4, b0[k]);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) reds_add(sa[k] + 8, log_top_word(b1[k], o0[k], b0[k], o[k], a[k]));
}
// log-scale value outside the fast path's reach
static __device__ __noinline__ void acc3_slow(uint32_t sa, float v, float mult, double* S1g, double* S2g) {
  if (v == 0.0f) return;
  const float t = v * mult;
  if (in_window_log(t)) { acc3_word(sa, __float2uint_rz(t)); return; }
  const double d = (double)v;                                      // outside the window, negative, NaN
  atomicAdd(S1g, d);
  atomicAdd(S2g, d * d);
}

// 2^23 <= t < 2^42: an exact integer of at most two words
__device__ __forceinline__ bool in_window_wide(float t) {
  return (__float_as_uint(t) - 0x4B000000u) < 0x09800000u;       // 2^42 = 0x54800000
}

// acc_quad for two-word a (a < 2^42, so a * a < 2^84): S1 in (w0, w1), S2 in (s0, s1, s2)
__device__ __forceinline__ void acc_quad_wide(uint32_t base, const uint32_t (&so)[4],
                                              const unsigned long long (&a)[4]) {
  uint32_t sa[4], o[4], o0[4], q0[4], q1[4], q2[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) { sa[k] = base + so[k]; o[k] = atoms_add(sa[k], (uint32_t)a[k]); }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const unsigned long long plo = a[k] * a[k], phi = __umul64hi(a[k], a[k]);   // phi < 2^20
    q0[k] = (uint32_t)plo; q1[k] = (uint32_t)(plo >> 32); q2[k] = (uint32_t)phi;
    o0[k] = atoms_add(sa[k] + 8, q0[k]);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const uint32_t hi = (uint32_t)(a[k] >> 32) + carry_of(o[k], (uint32_t)a[k]);
    if (hi) reds_add(sa[k] + 4, hi);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const unsigned long long m = (unsigned long long)q1[k] + carry_of(o0[k], q0[k]);
    q1[k] = (uint32_t)m;
    q2[k] += (uint32_t)(m >> 32);
    o[k] = atoms_add(sa[k] + 12, q1[k]);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const uint32_t top = q2[k] + carry_of(o[k], q1[k]);
    if (top) reds_add(sa[k] + 16, top);
  }
}

// any other value: wide a (2^32 <= a < 2^42), or outside the integer window -> global sums
static __device__ __noinline__ void acc_slow(uint32_t sa, float v, float mult, double* S1g, double* S2g) {
  if (v == 0.0f) return;
  const float t = v * mult;
  if (in_window(t)) { acc_word(sa, __float2uint_rz(t)); return; }
  if (t >= 4294967296.0f && t < 4398046511104.0f) {               // [2^32, 2^42)
    const unsigned long long a = __float2ull_rz(t);
    const uint32_t a0 = (uint32_t)a, a1 = (uint32_t)(a >> 32);
    const uint32_t o = atoms_add(sa, a0);
    reds_add(sa + 4, a1 + ((o + a0 < o) ? 1u : 0u));
    const unsigned long long plo = a * a, phi = __umul64hi(a, a);  // phi < 2^20
    const uint32_t q0 = (uint32_t)plo, q1 = (uint32_t)(plo >> 32), q2 = (uint32_t)phi;
    const uint32_t o0 = atoms_add(sa + 8, q0);
    const unsigned long long m = (unsigned long long)q1 + ((o0 + q0 < o0) ? 1u : 0u);
    const uint32_t m0 = (uint32_t)m;
    const uint32_t o1 = atoms_add(sa + 12, m0);
    reds_add(sa + 16, q2 + (uint32_t)(m >> 32) + ((o1 + m0 < o1) ? 1u : 0u));
    return;
  }
  const double d = (double)v;                                      // below the window, negative, NaN
  atomicAdd(S1g, d);
  atomicAdd(S2g, d * d);
}

// what the per-entry code needs to know about the CTA's accumulators
struct AccCtx {
  uint32_t sb_log, sb_lin;     // shared byte addresses of the two sets' tables
  float mult_log, mult_lin;
  int g0;
  uint32_t last_slot;          // Gt - 1
  double *S1log, *S2log, *S1lin, *S2lin;
};

// one entry, any value: normalise, log1p, accumulate; returns x''
// (MOM: moments-only pass, the value is x itself)
template <bool LOG, bool LIN, bool MOM>
__device__ __noinline__ float entry_any(const AccCtx& c, int j, float x, float scale) {
  const float xn = MOM ? x : __fmul_rn(x, scale);
  const float xl = MOM ? x : log1p_f32(xn);
  const uint32_t slot = min((uint32_t)(j - c.g0), c.last_slot);       // stays inside the table
  if (LOG) acc3_slow(c.sb_log + slot * (kLogWords * 4u), xl, c.mult_log, c.S1log + c.g0 + slot,
                     c.S2log + c.g0 + slot);
  if (LIN) acc_slow(c.sb_lin + slot * (kSetWords * 4u), xn, c.mult_lin, c.S1lin + c.g0 + slot,
                    c.S2lin + c.g0 + slot);
  return xl;
}

// A quad with at least one value outside the one-word window (out of line: keeps the hot path
// small).  All values at most two-word integers and x' >= 0.25 -> acc_quad_wide; else entry by
// entry.  valid_mask bit k: entry k belongs to the segment.
template <bool LOG, bool LIN, bool MOM>
__device__ __noinline__ float4 quad_rare(const AccCtx& c, int4 jv, float4 xv, float scale,
                                         uint32_t valid_mask, uint32_t spare_slot) {
  const int j[4] = {jv.x, jv.y, jv.z, jv.w};
  const float x[4] = {xv.x, xv.y, xv.z, xv.w};
  float xn[4], xl[4], tl[4], tn[4];
  bool ok = true;
  uint32_t slot[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const bool valid = (valid_mask >> k) & 1u;
    xn[k] = MOM ? x[k] : __fmul_rn(x[k], scale);
    xl[k] = MOM ? x[k] : log1p_ge_quarter(xn[k]);
    ok = ok && (MOM || xn[k] >= 0.25f || !valid);
    if (LOG) { tl[k] = xl[k] * c.mult_log; ok = ok && (in_window_log(tl[k]) || !valid); }
    if (LIN) { tn[k] = xn[k] * c.mult_lin; ok = ok && (in_window_wide(tn[k]) || !valid); }
    slot[k] = valid ? min((uint32_t)(j[k] - c.g0), c.last_slot) : spare_slot;
  }
  if (ok) {                     // only the linear-scale values need two words
    if (LOG) {
      uint32_t so[4], al[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        so[k] = slot[k] * (kLogWords * 4u);
        al[k] = ((valid_mask >> k) & 1u) ? __float2uint_rz(tl[k]) : 0u;
      }
      acc3_quad(c.sb_log, so, al);
    }
    if (LIN) {
      uint32_t so[4];
      unsigned long long an[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        so[k] = slot[k] * (kSetWords * 4u);
        an[k] = ((valid_mask >> k) & 1u) ? __float2ull_rz(tn[k]) : 0ull;
      }
      acc_quad_wide(c.sb_lin, so, an);
    }
  } else {
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if ((valid_mask >> k) & 1u) xl[k] = entry_any<LOG, LIN, MOM>(c, j[k], x[k], scale);
  }
  return make_float4(xl[0], xl[1], xl[2], xl[3]);
}

// fused.cu: integer totals of one set -> sums, mean, var
int launch_fused_finish(int32_t G, int64_t n_rows, int ddof, const FusedPlan* plan, int is_lin,
                        const unsigned long long* acc, double* S1, double* S2, double* mean, double* var,
                        cudaStream_t st);

}  // namespace rsc
