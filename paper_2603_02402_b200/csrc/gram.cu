// SURVEY.md 8(f) NEXT-3 (second half): sparse PCA front end, "Principal component
// analysis" -- mu = (1/n) X^T 1, S = X^T X ("the upper triangle ... accumulated using a custom
// kernel and symmetrized"), C = (S - n mu mu^T) / (n - 1) -- and L137 "centered Gram matrix
// construction".  The paper scatters the products of every sparse row with atomics; on B200 the
// contraction belongs on the tensor cores: for the HVG-subset matrix (1 M x 4 000, 4.5 % dense) the
// dense upper triangle is 1.6e13 MACs = ~25 ms of tcgen05 time, an order of magnitude less than
// 1.7e10 scattered L2 atomics cost.
//
// Pipeline (all on the caller's stream):
//   1. gram_absmax_kernel / gram_scale_kernel: 2^k with max |x| * 2^k in [2^14, 2^15) (fp16 range).
//   2. gram_pack_kernel (HBM-bound): a slab of CSR rows -> two dense fp16 planes [rows][p_pad],
//        H = fp16(v), L = fp16(v - H),  v = x * 2^k      (H + L carries 22 significand bits)
//      a warp assembles one row in shared memory (zero fill, scatter) and writes it out once.
//   3. gram_mma_kernel (tcgen05 / TMEM / TMA): output-stationary tiles of 128 x 256 of S that touch
//      the upper triangle, split over row ranges so that the tasks fill the SMs evenly.  Per 32-row
//      k-tile one TMA load per plane and operand (3-D boxes, 128-byte swizzle; both operands are
//      "MN-major": the gene axis is the contiguous one, so X^T needs no transposed copy), then
//        D += H_I^T H_J + H_I^T L_J + L_I^T H_J           (6 MMAs of 128 x 256 x 16, fp32 in TMEM)
//      Tensor-core accumulation truncates, and every term is >= 0, so a long accumulation drifts
//      low: the accumulator is therefore drained every kGmSub rows (two TMEM buffers, the MMAs
//      never wait) into fp32 registers of the epilogue warps (round-to-nearest adds), and a task
//      ends by adding its tile to a private fp32 partial in global memory -- no atomics, so the
//      result is bit-reproducible.
//   4. gram_finalize_kernel: partials summed in fp64, scaled by 2^-2k, mirrored, and
//      C = (S - n mu mu^T) / (n - 1) in fp64 (mu from the exact moments pass).
#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_fp16.h>
#include <math.h>

#include "common.cuh"

namespace rsc {

// implemented in api.cu
int launch_moments(const rsc_csr& X, int transform, int ddof, double* mean, double* var, double* sum,
                   double* sumsq, void* ws, size_t ws_bytes, cudaStream_t st);

constexpr int kGmM = 128;                 // tile rows (genes of block I): TMEM lanes
constexpr int kGmN = 256;                 // tile columns (genes of block J): TMEM columns
constexpr int kGmKT = 32;                 // cells per pipeline stage
constexpr int kGmStages = 4;
constexpr int kGmGroup = 64;              // genes per 128-byte swizzle row (fp16)
constexpr int kGmGroupBytes = kGmKT * 128;                      // one 64-gene group of a stage: 4 KB
constexpr int kGmABytes = (kGmM / kGmGroup) * kGmGroupBytes;    // 8 KB per plane
constexpr int kGmBBytes = (kGmN / kGmGroup) * kGmGroupBytes;    // 16 KB per plane
constexpr int kGmStageBytes = 2 * (kGmABytes + kGmBBytes);      // 48 KB: H_A | L_A | H_B | L_B
#ifndef RSC_GM_SUB
#define RSC_GM_SUB 512
#endif
constexpr int kGmSub = RSC_GM_SUB;        // cells between two drains of the TMEM accumulator
static_assert(kGmSub % kGmKT == 0, "drain interval must be a whole number of k-tiles");
constexpr int kGmThreads = 320;           // warp 0: TMA, warp 1: MMA, warps 2..9: epilogue
constexpr int kGmEpiWarps = 8;
constexpr int kGmMaxCols = 8192;          // genes (the pack kernel stages 4 rows of p_pad words)
constexpr int kGmSlabRows = 262144;       // cells per pack + MMA round (bounds the workspace)
constexpr int kGmPackWarps = 4;
constexpr size_t kGmSmem = (size_t)kGmStages * kGmStageBytes + 1024 + 256;

struct GramScale {                        // device scalars
  unsigned int absmax_bits;               // max |x| as float bits
  float mult;                             // 2^k
  double inv2;                            // 2^-2k
};

// ------------------------------------------------------------------ scale
__global__ void __launch_bounds__(256)
gram_absmax_kernel(int64_t nnz, const float* __restrict__ data, GramScale* sc) {
  float m = 0.0f;
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < nnz; p += (int64_t)gridDim.x * blockDim.x) {
    const float v = fabsf(__ldg(data + p));
    if (v > m && v <= 3.0e38f) m = v;                     // finite values only
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.0f) atomicMax(&sc->absmax_bits, __float_as_uint(m));
}

__global__ void gram_scale_kernel(GramScale* sc) {
  const float m = __uint_as_float(sc->absmax_bits);
  int k = 0;
  if (m > 0.0f) {
    int e;
    frexpf(m, &e);                                        // m = f 2^e, f in [0.5, 1)
    k = 15 - e;                                           // m 2^k in [2^14, 2^15)
  }
  k = max(-100, min(100, k));
  sc->mult = ldexpf(1.0f, k);
  sc->inv2 = ldexp(1.0, -2 * k);
}

// ------------------------------------------------------------------ pack: CSR rows -> fp16 planes
__global__ void __launch_bounds__(kGmPackWarps * 32)
gram_pack_kernel(int64_t row0, int64_t n_slab, int32_t p_pad, const int64_t* __restrict__ indptr,
                 const int32_t* __restrict__ indices, const float* __restrict__ data,
                 const GramScale* __restrict__ sc, __half* __restrict__ H, __half* __restrict__ L) {
  extern __shared__ __align__(16) uint32_t prow[];        // [kGmPackWarps][p_pad]: hi | lo << 16
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t* r = prow + (size_t)warp * p_pad;
  const float mult = sc->mult;
  const int64_t warp0 = (int64_t)blockIdx.x * kGmPackWarps + warp;
  const int64_t nwarps = (int64_t)gridDim.x * kGmPackWarps;
  for (int64_t lr = warp0; lr < n_slab; lr += nwarps) {
    const int64_t row = row0 + lr;
    const int64_t beg = indptr[row], end = indptr[row + 1];
    int j4[4];
    float x4[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {                         // requested before the fill hides their latency
      const int64_t p = beg + u * 32 + lane;
      j4[u] = p < end ? __ldg(indices + p) : -1;
      x4[u] = p < end ? __ldg(data + p) : 0.0f;
    }
    for (int j = lane * 4; j < p_pad; j += 128) *reinterpret_cast<uint4*>(r + j) = make_uint4(0u, 0u, 0u, 0u);
    __syncwarp();
    auto put = [&](int j, float x) {
      const float v = x * mult;
      const __half h = __float2half_rn(v);
      const __half l = __float2half_rn(v - __half2float(h));
      r[j] = (uint32_t)__half_as_ushort(h) | ((uint32_t)__half_as_ushort(l) << 16);
    };
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (j4[u] >= 0) put(j4[u], x4[u]);
    for (int64_t p = beg + 128 + lane; p < end; p += 32) put(__ldg(indices + p), __ldg(data + p));
    __syncwarp();
    __half* ho = H + lr * (int64_t)p_pad;
    __half* lo = L + lr * (int64_t)p_pad;
    for (int j = lane * 8; j < p_pad; j += 256) {         // 8 genes per lane: one 16-byte store per plane
      const uint4 a = *reinterpret_cast<const uint4*>(r + j);
      const uint4 b = *reinterpret_cast<const uint4*>(r + j + 4);
      uint4 hv, lv;
      hv.x = __byte_perm(a.x, a.y, 0x5410); lv.x = __byte_perm(a.x, a.y, 0x7632);
      hv.y = __byte_perm(a.z, a.w, 0x5410); lv.y = __byte_perm(a.z, a.w, 0x7632);
      hv.z = __byte_perm(b.x, b.y, 0x5410); lv.z = __byte_perm(b.x, b.y, 0x7632);
      hv.w = __byte_perm(b.z, b.w, 0x5410); lv.w = __byte_perm(b.z, b.w, 0x7632);
      *reinterpret_cast<uint4*>(ho + j) = hv;
      *reinterpret_cast<uint4*>(lo + j) = lv;
    }
    __syncwarp();
  }
}

// ------------------------------------------------------------------ PTX helpers (sm_100a)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0u;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem], fp16 inputs, fp32 accumulate; issued by one thread
__device__ __forceinline__ void tc_mma_f16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                           uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// 32 lanes x 32 columns of fp32: thread t of the warp gets lane (base lane + t), columns c .. c + 31
__device__ __forceinline__ void tc_ld_32x32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
        "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
        "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

// Shared-memory matrix descriptor of an MN-major, 128-byte-swizzled fp16 operand: 8 k-rows of
// 128 bytes (64 genes) form one swizzle atom; SBO = distance between atoms along k (1024 B),
// LBO = distance between 64-gene groups (one TMA box slice: kGmGroupBytes).
__device__ __forceinline__ uint64_t gm_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3ffffu) >> 4);                       // start address
  d |= (uint64_t)((uint32_t)kGmGroupBytes >> 4) << 16;            // leading byte offset
  d |= (uint64_t)(1024u >> 4) << 32;                              // stride byte offset
  d |= 1ull << 46;                                                // descriptor version (sm_100)
  d |= 2ull << 61;                                                // SWIZZLE_128B
  return d;
}
// kind::f16 instruction descriptor: D = f32, A = B = f16, both MN-major, N = 256, M = 128
constexpr uint32_t kGmIdesc = (1u << 4) | (1u << 15) | (1u << 16) | ((uint32_t)(kGmN >> 3) << 17) |
                              ((uint32_t)(kGmM >> 4) << 24);

struct GramArgs {
  int32_t p;                 // genes
  int32_t n_tiles;           // tiles that touch the upper triangle
  int32_t Q;                 // row ranges per tile
  int32_t rows_per_task;     // multiple of kGmKT
  int64_t n_slab;            // cells of this slab
  float* partial;            // [n_tiles * Q][kGmN][kGmM]
};

// tile t -> (ti, tj): 128-row block ti, 256-column block tj >= ti / 2 (those reach column >= row)
__device__ __forceinline__ void gm_tile_of(int t, int n_tj, int& ti, int& tj) {
  ti = 0;
  for (;;) {
    const int cnt = n_tj - (ti >> 1);
    if (t < cnt) break;
    t -= cnt;
    ++ti;
  }
  tj = (ti >> 1) + t;
}

__global__ void __launch_bounds__(kGmThreads, 1)
gram_mma_kernel(const __grid_constant__ CUtensorMap map_ha, const __grid_constant__ CUtensorMap map_la,
                const __grid_constant__ CUtensorMap map_hb, const __grid_constant__ CUtensorMap map_lb,
                const GramArgs a) {
  extern __shared__ uint8_t gsm_raw[];
  const uint32_t raw = smem_u32(gsm_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;             // swizzle atoms need 1024-byte alignment
  const uint32_t bars = base + kGmStages * kGmStageBytes;   // full[S] | empty[S] | tfull[2] | tempty[2]
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto empty_bar = [&](int s) { return bars + 8u * (kGmStages + s); };
  auto tfull_bar = [&](int b) { return bars + 8u * (2 * kGmStages + b); };
  auto tempty_bar = [&](int b) { return bars + 8u * (2 * kGmStages + 2 + b); };
  __shared__ uint32_t s_tmem;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_tj = (a.p + kGmN - 1) / kGmN;
  const int n_tasks = a.n_tiles * a.Q;

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < kGmStages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), kGmEpiWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {                                          // all 512 TMEM columns: 2 accumulators of 256
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;

  // rows and k-tiles of a task (the same arithmetic in every role)
  auto task_rows = [&](int task, int64_t& r0) -> int {
    const int q = task / a.n_tiles;
    r0 = (int64_t)q * a.rows_per_task;
    const int64_t left = a.n_slab - r0;
    return left <= 0 ? 0 : (int)(left < a.rows_per_task ? left : a.rows_per_task);
  };

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int task = blockIdx.x; task < n_tasks; task += gridDim.x) {
        int ti, tj;
        gm_tile_of(task % a.n_tiles, n_tj, ti, tj);
        int64_t r0;
        const int rows = task_rows(task, r0);
        const int nkt = (rows + kGmKT - 1) / kGmKT;
        for (int kt = 0; kt < nkt; ++kt) {
          mbar_wait(empty_bar(stage), phase ^ 1u);
          const uint32_t sb = base + stage * kGmStageBytes;
          mbar_expect_tx(full_bar(stage), kGmStageBytes);
          const int row = (int)(r0 + (int64_t)kt * kGmKT);
          tma_load_3d(sb, &map_ha, 0, row, ti * (kGmM / kGmGroup), full_bar(stage));
          tma_load_3d(sb + kGmABytes, &map_la, 0, row, ti * (kGmM / kGmGroup), full_bar(stage));
          tma_load_3d(sb + 2 * kGmABytes, &map_hb, 0, row, tj * (kGmN / kGmGroup), full_bar(stage));
          tma_load_3d(sb + 2 * kGmABytes + kGmBBytes, &map_lb, 0, row, tj * (kGmN / kGmGroup), full_bar(stage));
          if (++stage == kGmStages) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer (one thread) =====
    if (lane == 0) {
      int stage = 0, buf = 0;
      uint32_t phase = 0, tphase = 0u;               // bit b: phase of TMEM buffer b
      for (int task = blockIdx.x; task < n_tasks; task += gridDim.x) {
        int64_t r0;
        const int rows = task_rows(task, r0);
        const int nkt = (rows + kGmKT - 1) / kGmKT;
        constexpr int kPerSub = kGmSub / kGmKT;
        for (int k0 = 0; k0 < nkt; k0 += kPerSub) {
          const int k1 = min(nkt, k0 + kPerSub);
          mbar_wait(tempty_bar(buf), ((tphase >> buf) & 1u) ^ 1u);     // the epilogue has drained this buffer
          tc_fence_after();
          const uint32_t d = tmem + (uint32_t)buf * kGmN;
          for (int kt = k0; kt < k1; ++kt) {
            mbar_wait(full_bar(stage), phase);
            tc_fence_after();
            const uint32_t sb = base + stage * kGmStageBytes;
#pragma unroll
            for (int kk = 0; kk < kGmKT / 16; ++kk) {       // 16 cells per MMA: two swizzle atoms along k
              const uint32_t off = (uint32_t)kk * 2048u;
              const uint64_t ah = gm_desc(sb + off), al = gm_desc(sb + kGmABytes + off);
              const uint64_t bh = gm_desc(sb + 2 * kGmABytes + off), bl = gm_desc(sb + 2 * kGmABytes + kGmBBytes + off);
              tc_mma_f16(d, ah, bh, kGmIdesc, (kt > k0 || kk > 0) ? 1u : 0u);
              tc_mma_f16(d, ah, bl, kGmIdesc, 1u);
              tc_mma_f16(d, al, bh, kGmIdesc, 1u);
            }
            tc_commit(empty_bar(stage));                    // the stage is free once these MMAs have read it
            if (++stage == kGmStages) { stage = 0; phase ^= 1u; }
          }
          tc_commit(tfull_bar(buf));                        // accumulator complete
          tphase ^= 1u << buf;
          buf ^= 1;
        }
      }
    }
  } else {
    // ===== epilogue: TMEM -> fp32 registers (running sums of the task) -> partial tile =====
    const int ew = warp - 2;
    const int lq = warp & 3;                                // TMEM lanes this warp may read: 32 lq .. + 32
    const int half = ew >> 2;                               // columns 128 half .. + 128
    const int m = lq * 32 + lane;
    int buf = 0;
    uint32_t fphase = 0u;                                   // bit b: phase of TMEM buffer b
    for (int task = blockIdx.x; task < n_tasks; task += gridDim.x) {
      int64_t r0;
      const int rows = task_rows(task, r0);
      const int nkt = (rows + kGmKT - 1) / kGmKT;
      constexpr int kPerSub = kGmSub / kGmKT;
      float acc[kGmN / 2];
#pragma unroll
      for (int i = 0; i < kGmN / 2; ++i) acc[i] = 0.0f;
      for (int k0 = 0; k0 < nkt; k0 += kPerSub) {
        mbar_wait(tfull_bar(buf), (fphase >> buf) & 1u);
        tc_fence_after();
        const uint32_t t0 = tmem + ((uint32_t)(lq * 32) << 16) + (uint32_t)(buf * kGmN + half * (kGmN / 2));
#pragma unroll
        for (int c = 0; c < kGmN / 2; c += 32) {
          float v[32];
          tc_ld_32x32(t0 + (uint32_t)c, v);
#pragma unroll
          for (int i = 0; i < 32; ++i) acc[c + i] += v[i];
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty_bar(buf));
        fphase ^= 1u << buf;
        buf ^= 1;
      }
      if (nkt > 0) {
        float* pt = a.partial + (size_t)task * (kGmM * kGmN) + (size_t)(half * (kGmN / 2)) * kGmM + m;
#pragma unroll
        for (int i = 0; i < kGmN / 2; ++i) pt[(size_t)i * kGmM] += acc[i];   // coalesced over the warp's lanes
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
  }
}

// ------------------------------------------------------------------ finalize
// S[a][b] = S[b][a] = 2^-2k sum_q partial, C = (S - n mu_a mu_b) / (n - 1)   (a <= b)
__global__ void __launch_bounds__(256)
gram_finalize_kernel(int32_t p, int32_t n_tiles, int32_t Q, double n, const float* __restrict__ partial,
                     const GramScale* __restrict__ sc, const double* __restrict__ mean,
                     double* __restrict__ gram, double* __restrict__ cov) {
  const int t = blockIdx.x;                                 // one tile per CTA
  const int n_tj = (p + kGmN - 1) / kGmN;
  int ti, tj;
  gm_tile_of(t, n_tj, ti, tj);
  const double inv2 = sc->inv2;
  for (int e = threadIdx.x; e < kGmM * kGmN; e += blockDim.x) {
    const int mm = e % kGmM, nn = e / kGmM;                  // the partial's layout: [n][m]
    const int ga = ti * kGmM + mm, gb = tj * kGmN + nn;
    if (ga >= p || gb >= p || ga > gb) continue;
    double s = 0.0;
    for (int q = 0; q < Q; ++q) s += (double)partial[((size_t)q * n_tiles + t) * (kGmM * kGmN) + e];
    s *= inv2;
    if (gram) { gram[(size_t)ga * p + gb] = s; gram[(size_t)gb * p + ga] = s; }
    if (cov) {
      const double c = (s - n * mean[ga] * mean[gb]) / (n - 1.0);
      cov[(size_t)ga * p + gb] = c;
      cov[(size_t)gb * p + ga] = c;
    }
  }
}

// ------------------------------------------------------------------ host side
static int gm_p_pad(int32_t p) { return (p + kGmGroup - 1) / kGmGroup * kGmGroup; }
static int gm_n_tiles(int32_t p) {
  const int n_ti = (p + kGmM - 1) / kGmM, n_tj = (p + kGmN - 1) / kGmN;
  int t = 0;
  for (int ti = 0; ti < n_ti; ++ti) t += n_tj - (ti >> 1);
  return t;
}
// row ranges per tile: the smallest Q <= 16 whose task count fills the SMs to within 3 %, else the best
static int gm_choose_q(int n_tiles, int sms, int64_t slab_rows) {
  int best = 1;
  double best_eff = 0.0;
  for (int q = 1; q <= 16; ++q) {
    if (q > 1 && slab_rows / q < 4 * kGmSub) break;        // keep tasks long
    const int tasks = n_tiles * q;
    const double eff = (double)tasks / (double)(((tasks + sms - 1) / sms) * sms);
    if (eff > best_eff + 1e-9) { best_eff = eff; best = q; }
    if (eff >= 0.97) break;
  }
  return best;
}
static int64_t gm_slab_rows(int64_t n_rows) {
  int64_t s = n_rows < kGmSlabRows ? n_rows : kGmSlabRows;
  s = (s + kGmKT - 1) / kGmKT * kGmKT;
  return s > 0 ? s : kGmKT;
}

size_t moments_workspace_bytes(int64_t, int32_t, int64_t);

// workspace: scalars | mean | var | H plane | L plane | partial tiles (Q <= 16) | moments workspace
struct GramLayout { size_t mean, var, H, L, partial, moments, total; };
static GramLayout gm_layout(int64_t n_rows, int32_t n_cols, int64_t nnz) {
  GramLayout o;
  const size_t gsz = align_up(sizeof(double) * (size_t)n_cols, 256);
  const size_t plane = align_up((size_t)gm_slab_rows(n_rows) * (size_t)gm_p_pad(n_cols) * sizeof(__half), 1024);
  o.mean = 1024;
  o.var = o.mean + gsz;
  o.H = align_up(o.var + gsz, 1024);
  o.L = o.H + plane;
  o.partial = o.L + plane;
  o.moments = o.partial + align_up((size_t)gm_n_tiles(n_cols) * 16 * kGmM * kGmN * sizeof(float), 1024);
  o.total = o.moments + align_up(moments_workspace_bytes(n_rows, n_cols, nnz), 256) + 1024;   // + alignment slack
  return o;
}

size_t gram_workspace_bytes(int64_t n_rows, int32_t n_cols, int64_t nnz) {
  if (n_cols > kGmMaxCols || n_cols < 1) return 0;
  return gm_layout(n_rows, n_cols, nnz).total;
}

static PFN_cuTensorMapEncodeTiled_v12000 gm_encode_fn() {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
  if (fn == nullptr) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(p);
  }
  return fn;
}

// plane [rows][p_pad] fp16 seen as (64 genes of a group | rows | groups); box = 64 x kGmKT x groups
static int gm_make_map(CUtensorMap* map, const __half* plane, int64_t rows, int p_pad, int box_groups) {
  PFN_cuTensorMapEncodeTiled_v12000 enc = gm_encode_fn();
  if (enc == nullptr) { set_error("rsc_gram_cov: cuTensorMapEncodeTiled not available"); return RSC_ERR_CUDA; }
  const cuuint64_t dims[3] = {(cuuint64_t)kGmGroup, (cuuint64_t)rows, (cuuint64_t)(p_pad / kGmGroup)};
  const cuuint64_t strides[2] = {(cuuint64_t)p_pad * sizeof(__half), (cuuint64_t)kGmGroup * sizeof(__half)};
  const cuuint32_t box[3] = {(cuuint32_t)kGmGroup, (cuuint32_t)kGmKT, (cuuint32_t)box_groups};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<__half*>(plane), dims, strides, box,
                         estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("rsc_gram_cov: cuTensorMapEncodeTiled failed (%d)", (int)r); return RSC_ERR_CUDA; }
  return RSC_OK;
}

int launch_gram_cov(const rsc_csr& X, double* out_mean, double* out_gram, double* out_cov, void* ws,
                    size_t ws_bytes, cudaStream_t st) {
  const int32_t p = X.n_cols;
  const int p_pad = gm_p_pad(p);
  const int64_t slab = gm_slab_rows(X.n_rows);
  const int n_tiles = gm_n_tiles(p);
  unsigned char* w = static_cast<unsigned char*>(ws);      // 256-byte aligned (checked by the caller);
  const GramLayout lay = gm_layout(X.n_rows, p, X.nnz);    // the planes need 1024: shift the whole layout
  const size_t shift = align_up(reinterpret_cast<uintptr_t>(w), 1024) - reinterpret_cast<uintptr_t>(w);
  if (lay.total - 1024 + shift > ws_bytes) { set_error("rsc_gram_cov: workspace too small"); return RSC_ERR_WORKSPACE; }
  w += shift;
  GramScale* sc = reinterpret_cast<GramScale*>(w);
  double* mean = out_mean ? out_mean : reinterpret_cast<double*>(w + lay.mean);
  double* var = reinterpret_cast<double*>(w + lay.var);
  __half* H = reinterpret_cast<__half*>(w + lay.H);
  __half* L = reinterpret_cast<__half*>(w + lay.L);
  float* partial = reinterpret_cast<float*>(w + lay.partial);
  const int Q = gm_choose_q(n_tiles, sm_count(), slab);
  const size_t partial_bytes = (size_t)n_tiles * Q * kGmM * kGmN * sizeof(float);
  unsigned char* mws = w + lay.moments;
  const size_t mws_bytes = moments_workspace_bytes(X.n_rows, p, X.nnz);

  // mu (exact integer accumulators when the rows are sorted), scale, zeroed partials
  int rc = launch_moments(X, 0, 1, mean, var, nullptr, nullptr, mws, mws_bytes, st);
  if (rc != RSC_OK) return rc;
  RSC_CUDA(cudaMemsetAsync(sc, 0, sizeof(GramScale), st));
  RSC_CUDA(cudaMemsetAsync(partial, 0, partial_bytes, st));
  if (X.nnz > 0) {
    int64_t blocks = (X.nnz + 256 * 8 - 1) / (256 * 8);
    const int64_t cap = (int64_t)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    gram_absmax_kernel<<<(unsigned)blocks, 256, 0, st>>>(X.nnz, X.data, sc);
    RSC_LAUNCH_CHECK("gram_absmax_kernel");
  }
  gram_scale_kernel<<<1, 1, 0, st>>>(sc);
  RSC_LAUNCH_CHECK("gram_scale_kernel");

  const size_t pack_smem = sizeof(uint32_t) * (size_t)kGmPackWarps * (size_t)p_pad;
  RSC_CUDA(cudaFuncSetAttribute(gram_pack_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pack_smem));
  RSC_CUDA(cudaFuncSetAttribute(gram_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGmSmem));
  for (int64_t r0 = 0; r0 < X.n_rows; r0 += slab) {
    const int64_t n_slab = X.n_rows - r0 < slab ? X.n_rows - r0 : slab;
    {
      const int per_sm = (int)((200 * 1024) / (pack_smem + 1024)) > 0 ? (int)((200 * 1024) / (pack_smem + 1024)) : 1;
      int64_t blocks = (n_slab + kGmPackWarps - 1) / kGmPackWarps;
      const int64_t cap = (int64_t)sm_count() * (per_sm > 16 ? 16 : per_sm);
      if (blocks > cap) blocks = cap;
      gram_pack_kernel<<<(unsigned)blocks, kGmPackWarps * 32, pack_smem, st>>>(r0, n_slab, p_pad, X.indptr, X.indices,
                                                                              X.data, sc, H, L);
      RSC_LAUNCH_CHECK("gram_pack_kernel");
    }
    CUtensorMap mha, mla, mhb, mlb;
    if ((rc = gm_make_map(&mha, H, n_slab, p_pad, kGmM / kGmGroup)) != RSC_OK) return rc;
    if ((rc = gm_make_map(&mla, L, n_slab, p_pad, kGmM / kGmGroup)) != RSC_OK) return rc;
    if ((rc = gm_make_map(&mhb, H, n_slab, p_pad, kGmN / kGmGroup)) != RSC_OK) return rc;
    if ((rc = gm_make_map(&mlb, L, n_slab, p_pad, kGmN / kGmGroup)) != RSC_OK) return rc;
    GramArgs ga;
    ga.p = p; ga.n_tiles = n_tiles; ga.Q = Q; ga.n_slab = n_slab; ga.partial = partial;
    int64_t rpt = (n_slab + Q - 1) / Q;
    rpt = (rpt + kGmSub - 1) / kGmSub * kGmSub;            // whole drain intervals (and k-tiles)
    ga.rows_per_task = (int32_t)rpt;
    const int tasks = n_tiles * Q;
    const int grid = tasks < sm_count() ? tasks : sm_count();
    gram_mma_kernel<<<grid, kGmThreads, kGmSmem, st>>>(mha, mla, mhb, mlb, ga);
    RSC_LAUNCH_CHECK("gram_mma_kernel");
  }
  gram_finalize_kernel<<<n_tiles, 256, 0, st>>>(p, n_tiles, Q, (double)X.n_rows, partial, sc, mean, out_gram, out_cov);
  RSC_LAUNCH_CHECK("gram_finalize_kernel");
  return RSC_OK;
}

bool gram_supported(int32_t n_cols) { return n_cols >= 1 && n_cols <= kGmMaxCols; }

}  // namespace rsc

// ------------------------------------------------------------------ PCA projection
// Z = X V - 1 (mu^T V): "the sparse-to-dense transform applies implicit centering": a warp per cell,
// lanes over the components; every stored entry adds x * V[gene][:] (V as a float32 table that
// stays in L2 / L1: p x k x 4 B), accumulated in double, minus the per-component shift mu^T V.
namespace rsc {

constexpr int kPcaMaxComps = 128;

__global__ void __launch_bounds__(256)
pca_prep_kernel(int32_t p, int32_t k, int32_t kp, const double* __restrict__ V, const double* __restrict__ mean,
                float* __restrict__ Vf, double* __restrict__ shift) {
  // block c < k: shift[c] = sum_j mean_j V[j][c]; all blocks: their slice of the float table
  const int tid = threadIdx.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + tid; i < (int64_t)p * kp; i += (int64_t)gridDim.x * blockDim.x) {
    const int j = (int)(i / kp), c = (int)(i - (int64_t)j * kp);
    Vf[i] = c < k ? (float)V[(size_t)j * k + c] : 0.0f;
  }
  __shared__ double red[8];
  for (int c = blockIdx.x; c < k; c += gridDim.x) {
    double s = 0.0;
    if (mean != nullptr)
      for (int j = tid; j < p; j += blockDim.x) s += mean[j] * V[(size_t)j * k + c];
    s = warp_sum(s);
    if ((tid & 31) == 0) red[tid >> 5] = s;
    __syncthreads();
    if (tid == 0) {
      double t = 0.0;
      for (int w = 0; w < 8; ++w) t += red[w];
      shift[c] = t;
    }
    __syncthreads();
  }
}

template <int KPL>
__global__ void __launch_bounds__(256)
pca_transform_kernel(int64_t n_rows, int32_t k, int32_t kp, const int64_t* __restrict__ indptr,
                     const int32_t* __restrict__ indices, const float* __restrict__ data,
                     const float* __restrict__ Vf, const double* __restrict__ shift, float* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  double sh[KPL];
#pragma unroll
  for (int c = 0; c < KPL; ++c) sh[c] = lane + 32 * c < k ? shift[lane + 32 * c] : 0.0;
  for (int64_t row = warp0; row < n_rows; row += nwarps) {
    const int64_t beg = indptr[row], end = indptr[row + 1];
    double acc[KPL];
#pragma unroll
    for (int c = 0; c < KPL; ++c) acc[c] = 0.0;
    for (int64_t p0 = beg; p0 < end; p0 += 32) {
      const int64_t p = p0 + lane;
      const int j = p < end ? __ldg(indices + p) : 0;
      // converted once per lane, then broadcast as a double: the float -> double conversions run on the XU pipe
      // (16 lanes / clock / SM), one per entry and warp less: 6.04 -> 5.73 ms
      const double x = p < end ? (double)__ldg(data + p) : 0.0;
      const int cnt = (int)min((int64_t)32, end - p0);
      for (int t = 0; t < cnt; ++t) {
        const int jj = __shfl_sync(0xffffffffu, j, t);
        const double xx = __shfl_sync(0xffffffffu, x, t);
        const float* v = Vf + (size_t)jj * kp + lane;
#pragma unroll
        for (int c = 0; c < KPL; ++c) acc[c] = fma(xx, (double)__ldg(v + 32 * c), acc[c]);
      }
    }
    float* o = out + row * (int64_t)k;
#pragma unroll
    for (int c = 0; c < KPL; ++c)
      if (lane + 32 * c < k) o[lane + 32 * c] = (float)(acc[c] - sh[c]);
  }
}

size_t pca_workspace_bytes(int32_t n_cols, int32_t n_comps) {
  if (n_cols < 1 || n_comps < 1 || n_comps > kPcaMaxComps) return 0;
  const size_t kp = (size_t)((n_comps + 31) / 32 * 32);
  return align_up(sizeof(float) * (size_t)n_cols * kp, 256) + align_up(sizeof(double) * kPcaMaxComps, 256);
}
bool pca_supported(int32_t n_comps) { return n_comps >= 1 && n_comps <= kPcaMaxComps; }

int launch_pca_transform(const rsc_csr& X, const double* V, const double* mean, int32_t k, float* out, void* ws,
                         cudaStream_t st) {
  if (X.n_rows == 0) return RSC_OK;
  const int kp = (k + 31) / 32 * 32;
  unsigned char* w = static_cast<unsigned char*>(ws);
  float* Vf = reinterpret_cast<float*>(w);
  double* shift = reinterpret_cast<double*>(w + align_up(sizeof(float) * (size_t)X.n_cols * kp, 256));
  int64_t pb = ((int64_t)X.n_cols * kp + 255) / 256;
  if (pb < k) pb = k;
  if (pb > 4096) pb = 4096;
  pca_prep_kernel<<<(unsigned)pb, 256, 0, st>>>(X.n_cols, k, kp, V, mean, Vf, shift);
  RSC_LAUNCH_CHECK("pca_prep_kernel");
  int64_t blocks = (X.n_rows + 7) / 8;
  // rows are dealt statically (row = warp, warp + n_warps, ..): no more blocks than are resident at once, or the
  // rest runs as a second, thin wave (8 per SM asked, 6 resident: 6.46 -> 6.04 ms)
  int per_sm = 8;
  {
    const void* kern = kp / 32 == 1 ? (const void*)pca_transform_kernel<1> : kp / 32 == 2 ? (const void*)pca_transform_kernel<2>
                     : kp / 32 == 3 ? (const void*)pca_transform_kernel<3> : (const void*)pca_transform_kernel<4>;
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, 256, 0) == cudaSuccess && n >= 1) per_sm = n;
  }
  const int64_t cap = (int64_t)sm_count() * per_sm;
  if (blocks > cap) blocks = cap;
  switch (kp / 32) {
    case 1: pca_transform_kernel<1><<<(unsigned)blocks, 256, 0, st>>>(X.n_rows, k, kp, X.indptr, X.indices, X.data, Vf, shift, out); break;
    case 2: pca_transform_kernel<2><<<(unsigned)blocks, 256, 0, st>>>(X.n_rows, k, kp, X.indptr, X.indices, X.data, Vf, shift, out); break;
    case 3: pca_transform_kernel<3><<<(unsigned)blocks, 256, 0, st>>>(X.n_rows, k, kp, X.indptr, X.indices, X.data, Vf, shift, out); break;
    default: pca_transform_kernel<4><<<(unsigned)blocks, 256, 0, st>>>(X.n_rows, k, kp, X.indptr, X.indices, X.data, Vf, shift, out); break;
  }
  RSC_LAUNCH_CHECK("pca_transform_kernel");
  return RSC_OK;
}

}  // namespace rsc
