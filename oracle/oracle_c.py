"""CPU ORACLE, C / OpenMP twin (ctypes wrapper) -- test infrastructure, NOT a product path.

Row-parallel C restatement (oracle/oracle_c.c) of the oracle_np functions whose cost grows with
the number of stored entries, for the large BASELINE.json configurations and for the all-cores
CPU baseline of bench.py.  Same definitions, same float64 / int64 arithmetic as
oracle_np; pinned element-wise against it in tests/test_oracle_c.py.  The G-sized steps (HVG
selection) stay in oracle_np.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this module.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build
from . import oracle_np as _np_oracle

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        i64p, i32p, f32p, f64p, u8p = (C.POINTER(C.c_int64), C.POINTER(C.c_int32), C.POINTER(C.c_float),
                                       C.POINTER(C.c_double), C.POINTER(C.c_uint8))
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_qc.argtypes = [C.c_int64, C.c_int32, i64p, i32p, f32p, u8p, i64p, i32p, i64p, f32p, i64p, i64p]
        L.orc_normalize_log1p.argtypes = [C.c_int64, i64p, f32p, i64p, C.c_double, f32p, f32p]
        L.orc_gene_sums.argtypes = [C.c_int64, C.c_int32, i64p, i32p, f32p, C.c_int, f64p, f64p, f64p]
        L.orc_gene_sqdev.argtypes = [C.c_int64, C.c_int32, i64p, i32p, f32p, C.c_int, f64p, f64p]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(t: int) -> None:
    lib().orc_set_num_threads(int(t))


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def _csr(indptr, indices, data):
    return (np.ascontiguousarray(indptr, np.int64), np.ascontiguousarray(indices, np.int32),
            np.ascontiguousarray(data, np.float32))


def qc_metrics(indptr, indices, data, n_genes: int, gene_flags=None, gene_acc=None) -> dict:
    """oracle_np.qc_metrics (Q1..Q4).  gene_acc = (gene_n_cells i64, gene_total i64) lets a caller
    walking the matrix in row chunks accumulate the per-gene outputs across calls."""
    ip, ix, x = _csr(indptr, indices, data)
    n = ip.shape[0] - 1
    fl = None if gene_flags is None else np.ascontiguousarray(np.asarray(gene_flags) != 0, np.uint8)
    ct = np.zeros(n, np.int64); cn = np.zeros(n, np.int32); cf = np.zeros(n, np.int64)
    pct = np.zeros(n, np.float32)
    gn, gt = gene_acc if gene_acc is not None else (np.zeros(n_genes, np.int64), np.zeros(n_genes, np.int64))
    lib().orc_qc(n, n_genes, _p(ip, C.c_int64), _p(ix, C.c_int32), _p(x, C.c_float), _p(fl, C.c_uint8),
                 _p(ct, C.c_int64), _p(cn, C.c_int32), _p(cf, C.c_int64), _p(pct, C.c_float),
                 _p(gn, C.c_int64), _p(gt, C.c_int64))
    return dict(cell_total_i64=ct, cell_total_f32=ct.astype(np.float32), cell_n_genes=cn,
                cell_flag_total_i64=cf, cell_flag_pct=pct, gene_n_cells=gn.astype(np.int32),
                gene_total_i64=gt)


def normalize_log1p(indptr, data, target_sum: float, cell_total_i64, want_norm=True, want_log=True):
    """oracle_np.normalize_total followed by oracle_np.log1p: returns (x' f32 or None, x'' f32 or None)."""
    ip = np.ascontiguousarray(indptr, np.int64)
    x = np.ascontiguousarray(data, np.float32)
    tot = np.ascontiguousarray(cell_total_i64, np.int64)
    xn = np.empty_like(x) if want_norm else None
    xl = np.empty_like(x) if want_log else None
    lib().orc_normalize_log1p(ip.shape[0] - 1, _p(ip, C.c_int64), _p(x, C.c_float), _p(tot, C.c_int64),
                              float(target_sum), _p(xn, C.c_float), _p(xl, C.c_float))
    return xn, xl


def gene_sums(indptr, indices, data, n_genes: int, transform: int = 0, acc=None):
    """S1_j = sum v, S2_j = sum v^2, stored_j; acc = (S1, S2, stored) accumulates across row chunks."""
    ip, ix, x = _csr(indptr, indices, data)
    s1, s2, st = acc if acc is not None else (np.zeros(n_genes), np.zeros(n_genes), np.zeros(n_genes))
    lib().orc_gene_sums(ip.shape[0] - 1, n_genes, _p(ip, C.c_int64), _p(ix, C.c_int32), _p(x, C.c_float),
                        int(transform), _p(s1, C.c_double), _p(s2, C.c_double), _p(st, C.c_double))
    return s1, s2, st


def gene_sqdev(indptr, indices, data, n_genes: int, mean, transform: int = 0, acc=None):
    """SS_j = sum over stored entries of (v - mean_j)^2; acc accumulates across row chunks."""
    ip, ix, x = _csr(indptr, indices, data)
    ss = acc if acc is not None else np.zeros(n_genes)
    m = np.ascontiguousarray(mean, np.float64)
    lib().orc_gene_sqdev(ip.shape[0] - 1, n_genes, _p(ip, C.c_int64), _p(ix, C.c_int32), _p(x, C.c_float),
                         int(transform), _p(m, C.c_double), _p(ss, C.c_double))
    return ss


def moments_from(n: int, s1, stored, ss, ddof: int = 1):
    """mean and the two-pass variance of oracle_np.gene_moments from its three sums."""
    mean = s1 / np.float64(n) if n > 0 else np.zeros_like(s1)
    with np.errstate(divide="ignore", invalid="ignore"):
        var = (ss + (np.float64(n) - stored) * mean * mean) / np.float64(n - ddof)
    return mean, var


def gene_moments(indptr, indices, data, n_genes: int, transform: int = 0, ddof: int = 1):
    """oracle_np.gene_moments (M1): (mean, var, S1, S2), two passes."""
    n = len(indptr) - 1
    s1, s2, st = gene_sums(indptr, indices, data, n_genes, transform)
    mean = s1 / np.float64(n) if n > 0 else np.zeros(n_genes)
    ss = gene_sqdev(indptr, indices, data, n_genes, mean, transform)
    mean, var = moments_from(n, s1, st, ss, ddof)
    return mean, var, s1, s2


def preprocess_chain(indptr, indices, data, n_genes, gene_flags, target_sum, n_top, n_bins=20, ddof=1,
                     hvg_on="linear") -> dict:
    """oracle_np.preprocess_chain with the nnz-sized steps in C (composition only)."""
    qc = qc_metrics(indptr, indices, data, n_genes, gene_flags)
    xn, xl = normalize_log1p(indptr, data, target_sum, qc["cell_total_i64"])
    mean_log, var_log, _, _ = gene_moments(indptr, indices, xl, n_genes, 0, ddof)
    mean_lin, var_lin, _, _ = gene_moments(indptr, indices, xn, n_genes, 0, ddof)
    if hvg_on == "linear":
        hv = _np_oracle.hvg_select(mean_lin, var_lin, n_top, n_bins)
    else:
        hv = _np_oracle.hvg_select(mean_log, var_log, n_top, n_bins)
    return dict(qc=qc, x_norm=xn, x_log=xl, mean_log=mean_log, var_log=var_log, mean_lin=mean_lin,
                var_lin=var_lin, hvg=hv)
