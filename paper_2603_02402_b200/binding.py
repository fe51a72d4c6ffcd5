"""Thin ctypes binding of librsc_b200 (include/rsc.h).

Argument marshalling only: every step of the path runs inside the CUDA library.
PyTorch provides device memory and streams, nothing else.  There is NO CPU
fallback: if the shared library is missing, or no CUDA device is present, the
calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "librsc_b200.so")

RSC_OK = 0
RSC_ERR_INVALID_ARG = -1
RSC_ERR_WORKSPACE = -2
RSC_ERR_CUDA = -3
RSC_ERR_UNSUPPORTED = -4
RSC_CSR_SORTED = 1
RSC_MOMENTS_LOG = 1
RSC_MOMENTS_LIN = 2
RSC_MOMENTS_FP64_ACC = 4
RSC_SPLIT_WIDTH = 1024
RSC_HVG_SEURAT_LOG = 1

EXPORTS = [
    "rsc_last_error", "rsc_version", "rsc_kernel_launch_count",
    "rsc_row_splits_count", "rsc_row_splits", "rsc_set_option",
    "rsc_qc_metrics_workspace_bytes", "rsc_qc_metrics", "rsc_qc_metrics_splits",
    "rsc_moments_split_blocks",
    "rsc_normalize_total", "rsc_log1p",
    "rsc_gene_moments_workspace_bytes", "rsc_gene_moments",
    "rsc_normalize_log1p_moments_workspace_bytes", "rsc_normalize_log1p_moments",
    "rsc_moments_finalize",
    "rsc_hvg_select_workspace_bytes", "rsc_hvg_select",
    "rsc_hvg_select_no_alloc_max_genes", "rsc_hvg_select_no_alloc",
    "rsc_filter_masks", "rsc_subset_csr_workspace_bytes", "rsc_subset_csr_plan", "rsc_subset_csr_fill",
    "rsc_scale_dense_workspace_bytes", "rsc_scale_dense", "rsc_hvg_cutoffs",
    "rsc_gram_cov_workspace_bytes", "rsc_gram_cov", "rsc_pca_transform_workspace_bytes", "rsc_pca_transform",
    "rsc_hvg_select_cell_ranger_workspace_bytes", "rsc_hvg_select_cell_ranger", "rsc_hvg_merge_batches",
    "rsc_preprocess_workspace_bytes", "rsc_preprocess",
    "rsc_preprocess_host_workspace_bytes", "rsc_preprocess_host",
]


class RscError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"librsc_b200 error {code}: {msg}")
        self.code = code


class rsc_csr(C.Structure):
    _fields_ = [("n_rows", C.c_int64), ("n_cols", C.c_int32), ("flags", C.c_int32),
                ("nnz", C.c_int64), ("indptr", C.c_void_p), ("indices", C.c_void_p),
                ("data", C.c_void_p)]


_OUT_FIELDS = ["cell_total_i64", "cell_total_f32", "cell_n_genes", "cell_flag_total_i64",
               "cell_flag_pct", "gene_n_cells", "gene_total_i64", "mean_log", "var_log",
               "mean_lin", "var_lin", "hvg_mean_t", "hvg_disp", "hvg_disp_norm", "hvg_bin",
               "hvg_mask", "hvg_indices", "hvg_count"]


class rsc_outputs(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in _OUT_FIELDS]


class rsc_filter_params(C.Structure):
    _fields_ = [("min_genes", C.c_int32), ("min_cells", C.c_int32), ("min_counts", C.c_int64),
                ("min_gene_counts", C.c_int64), ("max_pct_flag", C.c_float), ("pad", C.c_int32)]


class rsc_params(C.Structure):
    _fields_ = [("target_sum", C.c_float), ("n_top", C.c_int32), ("n_bins", C.c_int32),
                ("ddof", C.c_int32), ("which_moments", C.c_int32), ("hvg_on_linear", C.c_int32),
                ("hvg_flags", C.c_int32)]


_lib = None


def lib() -> C.CDLL:
    """Load librsc_b200.so (raises if it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RscError(RSC_ERR_UNSUPPORTED,
                       f"{LIB_PATH} not found: run `python -m paper_2603_02402_b200.build` "
                       "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.rsc_last_error.restype = C.c_char_p
    L.rsc_version.restype = C.c_char_p
    L.rsc_kernel_launch_count.restype = C.c_uint64
    for name in EXPORTS:
        f = getattr(L, name)
        if name.endswith("_workspace_bytes") or name == "rsc_row_splits_count":
            f.restype = C.c_size_t
        elif name not in ("rsc_last_error", "rsc_version", "rsc_kernel_launch_count"):
            f.restype = C.c_int
    p, i32, i64, sz, flt = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t, C.c_float
    L.rsc_qc_metrics_workspace_bytes.argtypes = [i64, i32, i64]
    L.rsc_gene_moments_workspace_bytes.argtypes = [i64, i32, i64]
    L.rsc_normalize_log1p_moments_workspace_bytes.argtypes = [i64, i32, i64]
    L.rsc_hvg_select_workspace_bytes.argtypes = [i32, i32]
    L.rsc_subset_csr_workspace_bytes.argtypes = [i64, i32]
    L.rsc_scale_dense_workspace_bytes.argtypes = [i32]
    L.rsc_hvg_select_cell_ranger_workspace_bytes.argtypes = [i32]
    L.rsc_hvg_select_cell_ranger.argtypes = [i32, p, p, i32, p, p, p, p, p, p, p, sz, p]
    L.rsc_hvg_merge_batches.argtypes = [i32, i32, p, p, i32, p, p, p, p, p, p]
    L.rsc_pca_transform_workspace_bytes.argtypes = [i32, i32]
    L.rsc_pca_transform.argtypes = [p, p, p, i32, p, p, sz, p]
    L.rsc_gram_cov_workspace_bytes.argtypes = [i64, i32, i64]
    L.rsc_gram_cov.argtypes = [p, p, p, p, p, sz, p]
    L.rsc_hvg_cutoffs.argtypes = [i32, p, p, C.c_double, C.c_double, C.c_double, C.c_double, p, p, p, p]
    L.rsc_scale_dense.argtypes = [p, p, p, flt, C.c_int, p, p, sz, p]
    L.rsc_filter_masks.argtypes = [i64, i32, p, p, p, p, p, p, p, p, p]
    L.rsc_subset_csr_plan.argtypes = [p, p, p, p, p, p, sz, p]
    L.rsc_subset_csr_fill.argtypes = [p, p, p, p, p, sz, p]
    L.rsc_preprocess_workspace_bytes.argtypes = [i64, i32, i64, i32]
    L.rsc_preprocess_host_workspace_bytes.argtypes = [i64, i32, i64, i32]
    L.rsc_set_option.argtypes = [C.c_char_p, C.c_longlong]
    L.rsc_row_splits_count.argtypes = [i64, i32]
    L.rsc_row_splits.argtypes = [p, p, p]
    L.rsc_qc_metrics.argtypes = [p] + [p] * 9 + [p, sz, p]
    L.rsc_qc_metrics_splits.argtypes = [p] + [p] * 9 + [p, i32, p, sz, p]
    L.rsc_moments_split_blocks.argtypes = [i32, C.c_int, p, i32]
    L.rsc_moments_split_blocks.restype = i32
    L.rsc_normalize_total.argtypes = [p, flt, p, p, p]
    L.rsc_log1p.argtypes = [p, p]
    L.rsc_gene_moments.argtypes = [p, C.c_int, C.c_int, p, p, p, p, p, sz, p]
    L.rsc_normalize_log1p_moments.argtypes = [p, flt, p, p, p, C.c_int, C.c_int, p, p, p, p, p, p, sz, p]
    L.rsc_moments_finalize.argtypes = [i32, i64, C.c_int, p, p, p, p, p]
    L.rsc_hvg_select.argtypes = [i32, p, p, i32, i32, C.c_int, p, p, p, p, p, p, p, p, sz, p]
    L.rsc_hvg_select_no_alloc.argtypes = [i32, p, p, i32, i32, C.c_int, p, p, p, p, p, p, p, p]
    L.rsc_hvg_select_no_alloc_max_genes.argtypes = []
    L.rsc_hvg_select_no_alloc_max_genes.restype = i32
    L.rsc_preprocess.argtypes = [p, p, p, p, p, sz, p]
    L.rsc_preprocess_host.argtypes = [p, p, p, p, p, p, sz, p]
    _lib = L
    return L


def _check(rc: int):
    if rc != RSC_OK:
        raise RscError(rc, lib().rsc_last_error().decode())


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _ws(nbytes: int, device, stream=None) -> torch.Tensor:
    # torch's caching allocator returns 512-byte aligned blocks.  A temporary used by kernels
    # queued on a stream other than the current one is recorded on that stream, so the allocator
    # does not hand the block out again before those kernels have run.
    t = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)
    if stream is not None and t.is_cuda:
        t.record_stream(stream)
    return t


@dataclass
class Csr:
    """CSR view over torch tensors (device tensors for every call except *_host)."""
    indptr: torch.Tensor    # int64 [n_rows + 1]
    indices: torch.Tensor   # int32 [nnz]
    data: torch.Tensor      # float32 [nnz]
    n_cols: int
    sorted_indices: bool = True

    def __post_init__(self):
        assert self.indptr.dtype == torch.int64 and self.indices.dtype == torch.int32
        assert self.data.dtype == torch.float32
        assert self.indptr.is_contiguous() and self.indices.is_contiguous() and self.data.is_contiguous()

    @property
    def n_rows(self) -> int:
        return self.indptr.shape[0] - 1

    @property
    def nnz(self) -> int:
        return self.indices.shape[0]

    @property
    def device(self):
        return self.data.device

    def c_struct(self) -> rsc_csr:
        return rsc_csr(self.n_rows, self.n_cols, RSC_CSR_SORTED if self.sorted_indices else 0,
                       self.nnz, self.indptr.data_ptr(), self.indices.data_ptr(),
                       self.data.data_ptr())


def _need_cuda(X: Csr):
    if not X.data.is_cuda:
        raise RscError(RSC_ERR_INVALID_ARG, "device tensors required (no CPU fallback)")


def rsc_version() -> str:
    return lib().rsc_version().decode()


def rsc_kernel_launch_count() -> int:
    return int(lib().rsc_kernel_launch_count())


def rsc_set_option(key: str, value: int) -> None:
    _check(lib().rsc_set_option(key.encode(), int(value)))


def rsc_row_splits_count(n_rows: int, n_cols: int) -> int:
    return int(lib().rsc_row_splits_count(int(n_rows), int(n_cols)))


def rsc_row_splits(X: Csr, stream=None) -> torch.Tensor:
    """Row split table of a sorted CSR matrix (uint32 values in an int32 tensor)."""
    _need_cuda(X)
    out = torch.empty(max(1, rsc_row_splits_count(X.n_rows, X.n_cols)), dtype=torch.int32,
                      device=X.device)
    cs = X.c_struct()
    _check(lib().rsc_row_splits(C.byref(cs), _ptr(out), _stream(stream)))
    return out


def rsc_moments_split_blocks(n_cols: int, which_moments: int) -> list:
    """Block indices of the row split table that rsc_normalize_log1p_moments reads."""
    buf = (C.c_int32 * 80)()
    k = lib().rsc_moments_split_blocks(n_cols, which_moments, C.cast(buf, C.c_void_p), 80)
    return [int(buf[i]) for i in range(min(k, 80))]


def rsc_qc_metrics(X: Csr, gene_flags: Optional[torch.Tensor] = None, stream=None,
                   with_row_splits: bool = False, split_blocks: Optional[list] = None) -> dict:
    _need_cuda(X)
    L, dev, n, G = lib(), X.device, X.n_rows, X.n_cols
    out = dict(
        cell_total_i64=torch.empty(n, dtype=torch.int64, device=dev),
        cell_total_f32=torch.empty(n, dtype=torch.float32, device=dev),
        cell_n_genes=torch.empty(n, dtype=torch.int32, device=dev),
        cell_flag_total_i64=torch.empty(n, dtype=torch.int64, device=dev),
        cell_flag_pct=torch.empty(n, dtype=torch.float32, device=dev),
        gene_n_cells=torch.empty(G, dtype=torch.int32, device=dev),
        gene_total_i64=torch.empty(G, dtype=torch.int64, device=dev),
    )
    nb = L.rsc_qc_metrics_workspace_bytes(n, G, X.nnz)
    ws = _ws(nb, dev, stream)
    cs = X.c_struct()
    splits = None
    if with_row_splits and X.sorted_indices:
        splits = torch.empty(max(1, rsc_row_splits_count(n, G)), dtype=torch.int32, device=dev)
    outs = [_ptr(out[k]) for k in ("cell_total_i64", "cell_total_f32", "cell_n_genes",
                                   "cell_flag_total_i64", "cell_flag_pct", "gene_n_cells", "gene_total_i64")]
    if split_blocks:
        sb = (C.c_int32 * len(split_blocks))(*split_blocks)
        _check(L.rsc_qc_metrics_splits(C.byref(cs), _ptr(gene_flags), *outs, _ptr(splits),
                                       C.cast(sb, C.c_void_p), len(split_blocks), _ptr(ws), ws.numel(),
                                       _stream(stream)))
    else:
        _check(L.rsc_qc_metrics(C.byref(cs), _ptr(gene_flags), *outs, _ptr(splits), _ptr(ws), ws.numel(),
                                _stream(stream)))
    if splits is not None:
        out["row_splits"] = splits
    return out


def rsc_normalize_total(X: Csr, target_sum: float, cell_total_i64: Optional[torch.Tensor] = None,
                        return_scale: bool = False, stream=None):
    _need_cuda(X)
    scale = torch.empty(X.n_rows, dtype=torch.float32, device=X.device) if return_scale else None
    cs = X.c_struct()
    _check(lib().rsc_normalize_total(C.byref(cs), float(target_sum), _ptr(cell_total_i64),
                                     _ptr(scale), _stream(stream)))
    return scale


def rsc_log1p(X: Csr, stream=None) -> None:
    _need_cuda(X)
    cs = X.c_struct()
    _check(lib().rsc_log1p(C.byref(cs), _stream(stream)))


def rsc_gene_moments(X: Csr, transform: int = 0, ddof: int = 1, stream=None) -> dict:
    _need_cuda(X)
    L, dev, G = lib(), X.device, X.n_cols
    out = {k: torch.empty(G, dtype=torch.float64, device=dev) for k in ("mean", "var", "sum", "sumsq")}
    ws = _ws(L.rsc_gene_moments_workspace_bytes(X.n_rows, G, X.nnz), dev, stream)
    cs = X.c_struct()
    _check(L.rsc_gene_moments(C.byref(cs), transform, ddof, _ptr(out["mean"]), _ptr(out["var"]),
                              _ptr(out["sum"]), _ptr(out["sumsq"]), _ptr(ws), ws.numel(),
                              _stream(stream)))
    return out


def rsc_normalize_log1p_moments(X: Csr, target_sum: float, cell_total_i64: torch.Tensor,
                                gene_n_cells: Optional[torch.Tensor] = None,
                                which_moments: int = RSC_MOMENTS_LOG | RSC_MOMENTS_LIN,
                                ddof: int = 1, return_sums: bool = False, stream=None,
                                row_splits: Optional[torch.Tensor] = None) -> dict:
    _need_cuda(X)
    L, dev, G = lib(), X.device, X.n_cols
    out = {}
    if return_sums:
        out["sums"] = torch.zeros(4, G, dtype=torch.float64, device=dev)
    if which_moments & RSC_MOMENTS_LOG:
        out["mean_log"] = torch.empty(G, dtype=torch.float64, device=dev)
        out["var_log"] = torch.empty(G, dtype=torch.float64, device=dev)
    if which_moments & RSC_MOMENTS_LIN:
        out["mean_lin"] = torch.empty(G, dtype=torch.float64, device=dev)
        out["var_lin"] = torch.empty(G, dtype=torch.float64, device=dev)
    ws = _ws(L.rsc_normalize_log1p_moments_workspace_bytes(X.n_rows, G, X.nnz), dev, stream)
    cs = X.c_struct()
    _check(L.rsc_normalize_log1p_moments(
        C.byref(cs), float(target_sum), _ptr(cell_total_i64), _ptr(gene_n_cells), _ptr(row_splits),
        which_moments, ddof, _ptr(out.get("mean_log")), _ptr(out.get("var_log")), _ptr(out.get("mean_lin")),
        _ptr(out.get("var_lin")), _ptr(out.get("sums")), _ptr(ws), ws.numel(), _stream(stream)))
    return out


def rsc_moments_finalize(S1: torch.Tensor, S2: torch.Tensor, n_rows_total: int, ddof: int = 1,
                         stream=None) -> dict:
    if not S1.is_cuda:
        raise RscError(RSC_ERR_INVALID_ARG, "device tensors required (no CPU fallback)")
    assert S1.dtype == torch.float64 and S2.dtype == torch.float64 and S1.is_contiguous() and S2.is_contiguous()
    G = S1.shape[0]
    out = dict(mean=torch.empty(G, dtype=torch.float64, device=S1.device),
               var=torch.empty(G, dtype=torch.float64, device=S1.device))
    _check(lib().rsc_moments_finalize(G, int(n_rows_total), ddof, _ptr(S1), _ptr(S2),
                                      _ptr(out["mean"]), _ptr(out["var"]), _stream(stream)))
    return out


def rsc_hvg_select(gene_mean: torch.Tensor, gene_var: torch.Tensor, n_top: int, n_bins: int = 20,
                   flags: int = RSC_HVG_SEURAT_LOG, stream=None) -> dict:
    if not gene_mean.is_cuda:
        raise RscError(RSC_ERR_INVALID_ARG, "device tensors required (no CPU fallback)")
    assert gene_mean.dtype == torch.float64 and gene_var.dtype == torch.float64
    L, dev, G = lib(), gene_mean.device, gene_mean.shape[0]
    out = dict(
        mean_t=torch.empty(G, dtype=torch.float64, device=dev),
        disp=torch.empty(G, dtype=torch.float64, device=dev),
        disp_norm=torch.empty(G, dtype=torch.float64, device=dev),
        bin=torch.empty(G, dtype=torch.int32, device=dev),
        mask=torch.empty(G, dtype=torch.uint8, device=dev),
        indices=torch.full((G,), -1, dtype=torch.int32, device=dev),
        count=torch.zeros(1, dtype=torch.int32, device=dev),
    )
    ws = _ws(L.rsc_hvg_select_workspace_bytes(G, n_bins), dev, stream)
    _check(L.rsc_hvg_select(G, _ptr(gene_mean), _ptr(gene_var), n_top, n_bins, flags,
                            _ptr(out["mean_t"]), _ptr(out["disp"]), _ptr(out["disp_norm"]),
                            _ptr(out["bin"]), _ptr(out["mask"]), _ptr(out["indices"]),
                            _ptr(out["count"]), _ptr(ws), ws.numel(), _stream(stream)))
    return out


def rsc_hvg_select_no_alloc_max_genes() -> int:
    return int(lib().rsc_hvg_select_no_alloc_max_genes())


def rsc_hvg_select_no_alloc(gene_mean: torch.Tensor, gene_var: torch.Tensor, n_top: int, n_bins: int = 20,
                            flags: int = RSC_HVG_SEURAT_LOG, out: Optional[dict] = None, stream=None) -> dict:
    """rsc_hvg_select on the library's built-in scratch array: the C call allocates nothing.  `out`
    (tensors keyed as rsc_hvg_select returns them) lets the caller pre-allocate the outputs too."""
    if not gene_mean.is_cuda:
        raise RscError(RSC_ERR_INVALID_ARG, "device tensors required (no CPU fallback)")
    assert gene_mean.dtype == torch.float64 and gene_var.dtype == torch.float64
    L, dev, G = lib(), gene_mean.device, gene_mean.shape[0]
    if out is None:
        out = dict(
            mean_t=torch.empty(G, dtype=torch.float64, device=dev),
            disp=torch.empty(G, dtype=torch.float64, device=dev),
            disp_norm=torch.empty(G, dtype=torch.float64, device=dev),
            bin=torch.empty(G, dtype=torch.int32, device=dev),
            mask=torch.empty(G, dtype=torch.uint8, device=dev),
            indices=torch.full((G,), -1, dtype=torch.int32, device=dev),
            count=torch.zeros(1, dtype=torch.int32, device=dev),
        )
    _check(L.rsc_hvg_select_no_alloc(G, _ptr(gene_mean), _ptr(gene_var), n_top, n_bins, flags,
                                     _ptr(out.get("mean_t")), _ptr(out.get("disp")), _ptr(out.get("disp_norm")),
                                     _ptr(out.get("bin")), _ptr(out["mask"]), _ptr(out.get("indices")),
                                     _ptr(out["count"]), _stream(stream)))
    return out


_OUT_DTYPES = dict(
    cell_total_i64=torch.int64, cell_total_f32=torch.float32, cell_n_genes=torch.int32,
    cell_flag_total_i64=torch.int64, cell_flag_pct=torch.float32, gene_n_cells=torch.int32,
    gene_total_i64=torch.int64, mean_log=torch.float64, var_log=torch.float64,
    mean_lin=torch.float64, var_lin=torch.float64, hvg_mean_t=torch.float64,
    hvg_disp=torch.float64, hvg_disp_norm=torch.float64, hvg_bin=torch.int32,
    hvg_mask=torch.uint8, hvg_indices=torch.int32, hvg_count=torch.int32)


def _alloc_outputs(n: int, G: int, device, pin: bool = False) -> dict:
    out = {}
    for k, dt in _OUT_DTYPES.items():
        size = 1 if k == "hvg_count" else (n if k.startswith("cell_") else G)
        if pin:
            out[k] = torch.empty(size, dtype=dt).pin_memory()
        else:
            out[k] = torch.empty(size, dtype=dt, device=device)
    return out


def _params(target_sum, n_top, n_bins, ddof, which_moments, hvg_on_linear, hvg_flags) -> rsc_params:
    return rsc_params(float(target_sum), int(n_top), int(n_bins), int(ddof), int(which_moments),
                      1 if hvg_on_linear else 0, int(hvg_flags))


class Preprocessor:
    """rsc_preprocess with outputs and workspace allocated once (reusable across calls)."""

    def __init__(self, n_rows: int, n_cols: int, nnz: int, target_sum: float, n_top: int,
                 n_bins: int = 20, ddof: int = 1,
                 which_moments: int = RSC_MOMENTS_LOG | RSC_MOMENTS_LIN,
                 hvg_on_linear: bool = True, hvg_flags: int = RSC_HVG_SEURAT_LOG, device="cuda"):
        L = lib()
        self.params = _params(target_sum, n_top, n_bins, ddof, which_moments, hvg_on_linear, hvg_flags)
        self.out = _alloc_outputs(n_rows, n_cols, device)
        self.out_struct = rsc_outputs(*[self.out[k].data_ptr() for k in _OUT_FIELDS])
        self.ws = _ws(L.rsc_preprocess_workspace_bytes(n_rows, n_cols, nnz, n_bins), device)

    def run(self, X: Csr, gene_flags: Optional[torch.Tensor] = None, stream=None) -> dict:
        _need_cuda(X)
        cs = X.c_struct()
        _check(lib().rsc_preprocess(C.byref(cs), _ptr(gene_flags), C.byref(self.params),
                                    C.byref(self.out_struct), _ptr(self.ws), self.ws.numel(),
                                    _stream(stream)))
        return self.out

    def run_staged(self, X: Csr, gene_flags: Optional[torch.Tensor] = None, events=None,
                   stream=None) -> dict:
        """The same chain as `run`, issued as its three C-ABI calls (rsc_qc_metrics,
        rsc_normalize_log1p_moments, rsc_hvg_select) so that CUDA events can be recorded
        between the stages: events = [e0, e1, e2, e3] are recorded before QC, between the
        stages and after HVG, on the launching stream."""
        _need_cuda(X)
        L, o, p = lib(), self.out, self.params
        st = torch.cuda.current_stream() if stream is None else stream
        sp_ = C.c_void_p(st.cuda_stream)
        cs = X.c_struct()
        if not hasattr(self, "_stage_ws"):
            n, G, nnz = X.n_rows, X.n_cols, X.nnz
            self._stage_ws = [_ws(L.rsc_qc_metrics_workspace_bytes(n, G, nnz), X.device),
                              _ws(L.rsc_normalize_log1p_moments_workspace_bytes(n, G, nnz), X.device),
                              _ws(L.rsc_hvg_select_workspace_bytes(G, p.n_bins), X.device),
                              torch.empty(max(1, rsc_row_splits_count(n, G)), dtype=torch.int32,
                                          device=X.device) if X.sorted_indices else None]
        w0, w1, w2, sp = self._stage_ws
        if events:
            events[0].record(st)
        if not hasattr(self, "_need"):                     # split entries the fused pass reads
            nb = rsc_moments_split_blocks(X.n_cols, p.which_moments)
            nb = nb if 0 < len(nb) <= 32 else []
            self._need = (C.c_int32 * max(1, len(nb)))(*nb), len(nb)
        _check(L.rsc_qc_metrics_splits(C.byref(cs), _ptr(gene_flags), _ptr(o["cell_total_i64"]),
                                       _ptr(o["cell_total_f32"]), _ptr(o["cell_n_genes"]),
                                       _ptr(o["cell_flag_total_i64"]), _ptr(o["cell_flag_pct"]),
                                       _ptr(o["gene_n_cells"]), _ptr(o["gene_total_i64"]), _ptr(sp),
                                       C.cast(self._need[0], C.c_void_p), self._need[1],
                                       _ptr(w0), w0.numel(), sp_))
        if events:
            events[1].record(st)
        _check(L.rsc_normalize_log1p_moments(
            C.byref(cs), p.target_sum, _ptr(o["cell_total_i64"]), _ptr(o["gene_n_cells"]), _ptr(sp),
            p.which_moments, p.ddof, _ptr(o["mean_log"]), _ptr(o["var_log"]), _ptr(o["mean_lin"]),
            _ptr(o["var_lin"]), None, _ptr(w1), w1.numel(), sp_))
        if events:
            events[2].record(st)
        hm, hv = (o["mean_lin"], o["var_lin"]) if p.hvg_on_linear else (o["mean_log"], o["var_log"])
        _check(L.rsc_hvg_select(X.n_cols, _ptr(hm), _ptr(hv), p.n_top, p.n_bins, p.hvg_flags,
                                _ptr(o["hvg_mean_t"]), _ptr(o["hvg_disp"]), _ptr(o["hvg_disp_norm"]),
                                _ptr(o["hvg_bin"]), _ptr(o["hvg_mask"]), _ptr(o["hvg_indices"]),
                                _ptr(o["hvg_count"]), _ptr(w2), w2.numel(), sp_))
        if events:
            events[3].record(st)
        return self.out


def rsc_preprocess(X: Csr, gene_flags, target_sum, n_top, n_bins=20, ddof=1,
                   which_moments=RSC_MOMENTS_LOG | RSC_MOMENTS_LIN, hvg_on_linear=True,
                   hvg_flags=RSC_HVG_SEURAT_LOG, stream=None) -> dict:
    pp = Preprocessor(X.n_rows, X.n_cols, X.nnz, target_sum, n_top, n_bins, ddof, which_moments,
                      hvg_on_linear, hvg_flags, X.device)
    return pp.run(X, gene_flags, stream)


class HostPreprocessor:
    """rsc_preprocess_host: HOST CSR in, HOST results out, staged through a device workspace."""

    def __init__(self, n_rows: int, n_cols: int, nnz: int, target_sum: float, n_top: int,
                 n_bins: int = 20, ddof: int = 1,
                 which_moments: int = RSC_MOMENTS_LOG | RSC_MOMENTS_LIN,
                 hvg_on_linear: bool = True, hvg_flags: int = RSC_HVG_SEURAT_LOG, device="cuda",
                 copy_back_data: bool = False):
        L = lib()
        self.params = _params(target_sum, n_top, n_bins, ddof, which_moments, hvg_on_linear, hvg_flags)
        self.out = _alloc_outputs(n_rows, n_cols, "cpu", pin=True)
        self.out_struct = rsc_outputs(*[self.out[k].data_ptr() for k in _OUT_FIELDS])
        self.ws = _ws(L.rsc_preprocess_host_workspace_bytes(n_rows, n_cols, nnz, n_bins), device)
        self.data_out = torch.empty(nnz, dtype=torch.float32).pin_memory() if copy_back_data else None
        self.h2d_bytes = (n_rows + 1) * 8 + nnz * 8 + n_cols
        self.d2h_bytes = sum(t.numel() * t.element_size() for t in self.out.values()) + \
            (nnz * 4 if copy_back_data else 0)

    def run(self, hX: Csr, host_gene_flags: Optional[torch.Tensor] = None, stream=None) -> dict:
        if hX.data.is_cuda:
            raise RscError(RSC_ERR_INVALID_ARG, "rsc_preprocess_host takes HOST tensors")
        cs = hX.c_struct()
        _check(lib().rsc_preprocess_host(C.byref(cs), _ptr(host_gene_flags), C.byref(self.params),
                                         C.byref(self.out_struct), _ptr(self.data_out),
                                         _ptr(self.ws), self.ws.numel(), _stream(stream)))
        return self.out


# --------------------------------------------------------------------------- NEXT-1: filtering
def rsc_filter_masks(qc: dict, min_genes: int = 0, min_counts: int = 0,
                     max_pct_flag: float = float("inf"), min_cells: int = 0,
                     min_gene_counts: int = 0, stream=None):
    """uint8 keep-masks (cells, genes) from the outputs of rsc_qc_metrics."""
    n, G = qc["cell_n_genes"].numel(), qc["gene_n_cells"].numel()
    dev = qc["cell_n_genes"].device
    if dev.type != "cuda":
        raise RscError(RSC_ERR_INVALID_ARG, "rsc_filter_masks needs device tensors (no CPU fallback)")
    prm = rsc_filter_params(min_genes, min_cells, min_counts, min_gene_counts, max_pct_flag, 0)
    ck = torch.empty(n, dtype=torch.uint8, device=dev)
    gk = torch.empty(G, dtype=torch.uint8, device=dev)
    _check(lib().rsc_filter_masks(n, G, _ptr(qc["cell_n_genes"]), _ptr(qc["cell_total_i64"]),
                                  _ptr(qc["cell_flag_pct"]), _ptr(qc["gene_n_cells"]),
                                  _ptr(qc["gene_total_i64"]), C.byref(prm), _ptr(ck), _ptr(gk),
                                  _stream(stream)))
    return ck, gk


def rsc_subset_csr(X: Csr, keep_rows: Optional[torch.Tensor] = None,
                   keep_cols: Optional[torch.Tensor] = None, stream=None) -> Csr:
    """X[keep_rows][:, keep_cols] (uint8 masks or None) as a new device Csr: plan, one read of
    the three output sizes (the only synchronisation), allocation, fill."""
    _need_cuda(X)
    L, dev = lib(), X.device
    ws = _ws(L.rsc_subset_csr_workspace_bytes(X.n_rows, X.n_cols), dev, stream)
    out_indptr = torch.empty(X.n_rows + 1, dtype=torch.int64, device=dev)
    counts = torch.zeros(3, dtype=torch.int64, device=dev)
    cs = X.c_struct()
    _check(L.rsc_subset_csr_plan(C.byref(cs), _ptr(keep_rows), _ptr(keep_cols), _ptr(out_indptr),
                                 _ptr(counts), _ptr(ws), ws.numel(), _stream(stream)))
    if stream is not None:
        stream.synchronize()                               # .tolist() only waits for the CURRENT stream
    n_out, g_out, nnz_out = (int(v) for v in counts.tolist())
    out_indices = torch.empty(nnz_out, dtype=torch.int32, device=dev)
    out_data = torch.empty(nnz_out, dtype=torch.float32, device=dev)
    _check(L.rsc_subset_csr_fill(C.byref(cs), _ptr(keep_rows), _ptr(out_indices), _ptr(out_data),
                                 _ptr(ws), ws.numel(), _stream(stream)))
    return Csr(out_indptr[: n_out + 1], out_indices, out_data, max(g_out, 1), X.sorted_indices), g_out


# --------------------------------------------------------------------------- NEXT-3: scale
def rsc_scale_dense(X: Csr, gene_mean: torch.Tensor, gene_var: torch.Tensor,
                    max_value: Optional[float] = None, zero_center: bool = True, stream=None) -> torch.Tensor:
    """Dense float32 [n_rows, n_cols] z-scores (clipped to max_value if given)."""
    _need_cuda(X)
    L = lib()
    out = torch.empty((X.n_rows, X.n_cols), dtype=torch.float32, device=X.device)
    ws = _ws(L.rsc_scale_dense_workspace_bytes(X.n_cols), X.device, stream)
    cs = X.c_struct()
    _check(L.rsc_scale_dense(C.byref(cs), _ptr(gene_mean), _ptr(gene_var),
                             float(max_value) if max_value is not None else 0.0, int(bool(zero_center)),
                             _ptr(out), _ptr(ws), ws.numel(), _stream(stream)))
    return out


# --------------------------------------------------------------------------- NEXT-4 (part): cutoffs
def rsc_hvg_select_cell_ranger(gene_mean: torch.Tensor, gene_var: torch.Tensor, n_top: int, stream=None) -> dict:
    """Cell-ranger-flavour HVG selection from the moments of the normalised, non-logged matrix."""
    if not gene_mean.is_cuda:
        raise RscError(RSC_ERR_INVALID_ARG, "device tensors required (no CPU fallback)")
    assert gene_mean.dtype == torch.float64 and gene_var.dtype == torch.float64
    L, dev, G = lib(), gene_mean.device, gene_mean.shape[0]
    out = dict(disp=torch.empty(G, dtype=torch.float64, device=dev),
               disp_norm=torch.empty(G, dtype=torch.float64, device=dev),
               bin=torch.empty(G, dtype=torch.int32, device=dev),
               mask=torch.empty(G, dtype=torch.uint8, device=dev),
               indices=torch.full((G,), -1, dtype=torch.int32, device=dev),
               count=torch.zeros(1, dtype=torch.int32, device=dev))
    ws = _ws(L.rsc_hvg_select_cell_ranger_workspace_bytes(G), dev, stream)
    _check(L.rsc_hvg_select_cell_ranger(G, _ptr(gene_mean), _ptr(gene_var), n_top, _ptr(out["disp"]),
                                        _ptr(out["disp_norm"]), _ptr(out["bin"]), _ptr(out["mask"]),
                                        _ptr(out["indices"]), _ptr(out["count"]), _ptr(ws), ws.numel(),
                                        _stream(stream)))
    return out


def rsc_hvg_merge_batches(masks: torch.Tensor, disp_norm: torch.Tensor, n_top: int, stream=None) -> dict:
    """Merge per-batch HVG selections: masks uint8 [B, G], disp_norm float64 [B, G] (device)."""
    if not masks.is_cuda:
        raise RscError(RSC_ERR_INVALID_ARG, "device tensors required (no CPU fallback)")
    assert masks.dtype == torch.uint8 and disp_norm.dtype == torch.float64
    assert masks.is_contiguous() and disp_norm.is_contiguous() and masks.shape == disp_norm.shape
    Bn, G = masks.shape
    dev = masks.device
    out = dict(nbatches=torch.empty(G, dtype=torch.int32, device=dev),
               disp_norm_mean=torch.empty(G, dtype=torch.float64, device=dev),
               mask=torch.empty(G, dtype=torch.uint8, device=dev),
               indices=torch.full((G,), -1, dtype=torch.int32, device=dev),
               count=torch.zeros(1, dtype=torch.int32, device=dev))
    _check(lib().rsc_hvg_merge_batches(G, Bn, _ptr(masks), _ptr(disp_norm), n_top, _ptr(out["nbatches"]),
                                       _ptr(out["disp_norm_mean"]), _ptr(out["mask"]), _ptr(out["indices"]),
                                       _ptr(out["count"]), _stream(stream)))
    return out


def rsc_hvg_select_batched(X: Csr, batch_offsets, gene_flags, target_sum: float, n_top: int, n_bins: int = 20,
                           flavor: str = "seurat") -> dict:
    """Per-batch HVG over contiguous row ranges (batch b = rows batch_offsets[b] .. batch_offsets[b+1]):
    the chain runs once per batch on its row slice (x'' is written in place, so afterwards the whole
    matrix is log-normalised), the per-batch selections are merged by rsc_hvg_merge_batches.
    Marshalling only: every step is a C-ABI call."""
    _need_cuda(X)
    nb = len(batch_offsets) - 1
    masks = torch.empty(nb, X.n_cols, dtype=torch.uint8, device=X.device)
    zs = torch.empty(nb, X.n_cols, dtype=torch.float64, device=X.device)
    per_batch = []
    for b in range(nb):
        r0, r1 = int(batch_offsets[b]), int(batch_offsets[b + 1])
        p0, p1 = int(X.indptr[r0]), int(X.indptr[r1])
        Xb = Csr((X.indptr[r0:r1 + 1] - p0).contiguous(), X.indices[p0:p1], X.data[p0:p1], X.n_cols,
                 X.sorted_indices)
        o = rsc_preprocess(Xb, gene_flags, target_sum, n_top, n_bins, which_moments=RSC_MOMENTS_LOG | RSC_MOMENTS_LIN,
                           hvg_on_linear=True)
        if flavor == "cell_ranger":
            h = rsc_hvg_select_cell_ranger(o["mean_lin"], o["var_lin"], n_top)
            masks[b].copy_(h["mask"]); zs[b].copy_(h["disp_norm"])
        else:
            masks[b].copy_(o["hvg_mask"]); zs[b].copy_(o["hvg_disp_norm"])
        per_batch.append(o)
    out = rsc_hvg_merge_batches(masks, zs, n_top)
    out["batch_masks"], out["batch_disp_norm"], out["per_batch"] = masks, zs, per_batch
    return out


def rsc_pca_transform(X: Csr, V: torch.Tensor, gene_mean: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """PAPER.md:L95 Z = X V - 1 (mu^T V) as float32 [n_rows, n_comps]; V float64 [n_cols, n_comps]."""
    _need_cuda(X)
    assert V.is_cuda and V.dtype == torch.float64 and V.is_contiguous() and V.shape[0] == X.n_cols
    assert gene_mean is None or (gene_mean.dtype == torch.float64 and gene_mean.is_cuda)
    k = int(V.shape[1])
    out = torch.empty(X.n_rows, k, dtype=torch.float32, device=X.device)
    L = lib()
    ws = _ws(L.rsc_pca_transform_workspace_bytes(X.n_cols, k), X.device, stream)
    cs = X.c_struct()
    _check(L.rsc_pca_transform(C.byref(cs), _ptr(V), _ptr(gene_mean), k, _ptr(out), _ptr(ws), ws.numel(),
                               _stream(stream)))
    return out


def rsc_gram_cov(X: Csr, want_gram: bool = True, want_cov: bool = True, stream=None) -> dict:
    """PAPER.md:L95 mu, S = X^T X, C = (S - n mu mu^T) / (n - 1) on the tensor cores (float64 outputs)."""
    _need_cuda(X)
    L, dev, G = lib(), X.device, X.n_cols
    out = {"mean": torch.empty(G, dtype=torch.float64, device=dev)}
    if want_gram:
        out["gram"] = torch.empty(G, G, dtype=torch.float64, device=dev)
    if want_cov:
        out["cov"] = torch.empty(G, G, dtype=torch.float64, device=dev)
    ws = _ws(L.rsc_gram_cov_workspace_bytes(X.n_rows, G, X.nnz), dev, stream)
    cs = X.c_struct()
    _check(L.rsc_gram_cov(C.byref(cs), _ptr(out["mean"]), _ptr(out.get("gram")), _ptr(out.get("cov")),
                          _ptr(ws), ws.numel(), _stream(stream)))
    return out


def rsc_hvg_cutoffs(mean_t: torch.Tensor, disp_norm: torch.Tensor, min_mean: float = 0.0125,
                    max_mean: float = 3.0, min_disp: float = 0.5, max_disp: float = float("inf"),
                    stream=None) -> dict:
    """Threshold-based HVG selection from rsc_hvg_select's mean_t / disp_norm outputs."""
    if mean_t.device.type != "cuda":
        raise RscError(RSC_ERR_INVALID_ARG, "device tensors required (no CPU fallback)")
    G, dev = mean_t.numel(), mean_t.device
    out = dict(mask=torch.empty(G, dtype=torch.uint8, device=dev),
               indices=torch.empty(G, dtype=torch.int32, device=dev),
               count=torch.zeros(1, dtype=torch.int32, device=dev))
    _check(lib().rsc_hvg_cutoffs(G, _ptr(mean_t), _ptr(disp_norm), min_mean, max_mean, min_disp, max_disp,
                                 _ptr(out["mask"]), _ptr(out["indices"]), _ptr(out["count"]), _stream(stream)))
    return out
