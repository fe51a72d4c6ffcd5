"""paper_2603_02402_b200 — B200-native sparse-CSR single-cell preprocessing chain.

QC reductions -> normalize_total -> log1p -> per-gene moments -> Seurat-flavour HVG
selection (arxiv/paper_2603_02402), as hand-written sm_100a CUDA
kernels behind the C ABI of include/rsc.h.  `binding` is the ctypes layer; `synth`
is the seeded input generator (no method arithmetic); `build` compiles the library.
Importing the package does not load the CUDA library; the first call does, and it
raises if the library is missing (there is no CPU fallback).
"""
from .binding import (  # noqa: F401
    Csr, HostPreprocessor, Preprocessor, RscError,
    RSC_CSR_SORTED, RSC_HVG_SEURAT_LOG, RSC_MOMENTS_LIN, RSC_MOMENTS_LOG,
    rsc_gene_moments, rsc_hvg_select, rsc_log1p, rsc_moments_finalize, rsc_normalize_log1p_moments,
    rsc_normalize_total, rsc_preprocess, rsc_qc_metrics, rsc_version,
    rsc_filter_masks, rsc_subset_csr, rsc_scale_dense, rsc_gram_cov, rsc_pca_transform,
    rsc_hvg_select_cell_ranger, rsc_hvg_merge_batches, rsc_hvg_select_batched, rsc_hvg_cutoffs,
    rsc_hvg_select_no_alloc, rsc_hvg_select_no_alloc_max_genes,
)

__all__ = [
    "Csr", "HostPreprocessor", "Preprocessor", "RscError", "rsc_gene_moments", "rsc_hvg_select",
    "rsc_log1p", "rsc_moments_finalize", "rsc_normalize_log1p_moments", "rsc_normalize_total", "rsc_preprocess",
    "rsc_qc_metrics", "rsc_version", "rsc_filter_masks", "rsc_subset_csr", "rsc_scale_dense", "rsc_gram_cov", "rsc_pca_transform",
    "rsc_hvg_select_cell_ranger", "rsc_hvg_merge_batches", "rsc_hvg_select_batched", "rsc_hvg_cutoffs",
    "rsc_hvg_select_no_alloc", "rsc_hvg_select_no_alloc_max_genes",
]
