// rsc_hvg_select_no_alloc: rsc_hvg_select ("Highly variable gene selection is based on
// per-gene mean and variance", L39 "gene selection" on the device) for callers that can neither
// allocate device memory nor hand in a workspace: code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  The scratch the HVG kernels need (the transformed mean, the
// dispersion, the z-score and the bin id of every gene when the caller does not ask for them, plus
// the per-block extrema of the one-CTA kernel) lives in ONE file-scope device array of a fixed size:
//   * RSC_HVG_NO_ALLOC_MAX_GENES = 65 536 genes -> 2 MiB, held by every GPU that loads the library
//     until the process exits;
//   * the entry point rejects more genes with RSC_ERR_INVALID_ARG and calls no cudaMalloc / cudaFree
//     nor any allocating library routine (the kernels are the ones rsc_hvg_select launches);
//   * every call on a device shares the array.  The kernels write every scratch element before they
//     read it (nothing has to start at zero, so nothing is cleared), but two calls that OVERLAP on the
//     GPU (different streams, or graphs replayed concurrently) race on it: serialise them.
// In host code `g_hvg_scratch` is only a host-side stand-in for the symbol, not a device address;
// the address a kernel can use comes from cudaGetSymbolAddress, asked once per device with that
// device current (the array exists once per device).
#include <mutex>

#include "common.cuh"

namespace rsc {

constexpr int kNoAllocMaxGenes = RSC_HVG_NO_ALLOC_MAX_GENES;
constexpr size_t kNoAllocBytes = 2u << 20;                      // >= hvg_workspace_bytes(kNoAllocMaxGenes, *)
constexpr int kNoAllocMaxDevices = 64;

static __device__ __align__(256) unsigned char g_hvg_scratch[kNoAllocBytes];

static std::mutex g_na_mutex;
static void* g_na_ptr[kNoAllocMaxDevices];                      // device address of g_hvg_scratch, by device ordinal

// the device address of the scratch array on the CURRENT device (looked up once per device)
static int no_alloc_scratch(void** out) {
  int dev = -1;
  RSC_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoAllocMaxDevices) {
    set_error("rsc_hvg_select_no_alloc: device ordinal %d is beyond the %d this entry point tracks", dev,
              kNoAllocMaxDevices);
    return RSC_ERR_UNSUPPORTED;
  }
  std::lock_guard<std::mutex> lock(g_na_mutex);
  if (g_na_ptr[dev] == nullptr) {
    void* p = nullptr;
    RSC_CUDA(cudaGetSymbolAddress(&p, g_hvg_scratch));
    if (p == nullptr || (reinterpret_cast<uintptr_t>(p) & 255)) {
      set_error("rsc_hvg_select_no_alloc: the scratch array has no usable device address on device %d", dev);
      return RSC_ERR_CUDA;
    }
    g_na_ptr[dev] = p;
  }
  *out = g_na_ptr[dev];
  return RSC_OK;
}

}  // namespace rsc

extern "C" {

int32_t rsc_hvg_select_no_alloc_max_genes(void) { return rsc::kNoAllocMaxGenes; }

int rsc_hvg_select_no_alloc(int32_t n_genes, const double* gene_mean, const double* gene_var, int32_t n_top,
                            int32_t n_bins, int flags, double* out_mean_t, double* out_disp,
                            double* out_disp_norm, int32_t* out_bin, uint8_t* out_mask, int32_t* out_indices,
                            int32_t* out_count, void* stream) {
  using namespace rsc;
  RSC_CHECK_ARG(n_genes >= 1, "rsc_hvg_select_no_alloc: n_genes < 1");
  RSC_CHECK_ARG(n_genes <= kNoAllocMaxGenes,
                "rsc_hvg_select_no_alloc: n_genes = %d exceeds the built-in scratch (at most %d genes); "
                "use rsc_hvg_select with a caller-provided workspace", n_genes, kNoAllocMaxGenes);
  RSC_CHECK_ARG(gene_mean && gene_var, "rsc_hvg_select_no_alloc: gene_mean / gene_var are required");
  RSC_CHECK_ARG(n_top >= 1, "rsc_hvg_select_no_alloc: n_top < 1");
  RSC_CHECK_ARG(n_bins >= 1 && n_bins <= 4096, "rsc_hvg_select_no_alloc: n_bins must be in [1, 4096]");
  RSC_CHECK_ARG(out_mask && out_count, "rsc_hvg_select_no_alloc: out_mask / out_count are required");
  int rc = check_device();
  if (rc) return rc;
  if (hvg_workspace_bytes(n_genes, n_bins) > kNoAllocBytes) {      // cannot happen below the gene limit
    set_error("rsc_hvg_select_no_alloc: %zu bytes of scratch needed, %zu built in",
              hvg_workspace_bytes(n_genes, n_bins), kNoAllocBytes);
    return RSC_ERR_WORKSPACE;
  }
  void* scratch = nullptr;
  if ((rc = no_alloc_scratch(&scratch)) != RSC_OK) return rc;
  return launch_hvg(n_genes, gene_mean, gene_var, n_top, n_bins, flags, out_mean_t, out_disp, out_disp_norm,
                    out_bin, out_mask, out_indices, out_count, scratch, kNoAllocBytes,
                    static_cast<cudaStream_t>(stream));
}

}  // extern "C"
