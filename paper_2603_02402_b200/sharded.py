"""Row-sharded multi-GPU chain: one process per GPU, each holding a shard of the cells.

The paper scales out by partitioning the matrix "into chunks along the cell axis"
(Dask).  Here the same partitioning runs as one process per GPU over
`torch.distributed`: per-cell outputs, normalisation and log1p are independent per row; the
per-gene integer counts / totals and the double-precision sums S1, S2 need exactly ONE
exchange each — an all-reduce(sum) of a contiguous per-gene block (<= 36 k genes x 4
doubles ~ 1.2 MB, latency-bound on NVLink) — after which every rank finalises the moments
with the global cell count and runs the identical HVG selection.

`allreduce_gene_stats` is device-agnostic (it only packs, all-reduces and unpacks), so the
host-side logic is covered by world_size-2 gloo tests on CPU; the kernels are the same
single-GPU C-ABI calls.
"""
from __future__ import annotations

import ctypes as C
from typing import Dict, Optional

import torch
import torch.distributed as dist

from . import binding as B


def allreduce_gene_stats(int_stats: Dict[str, torch.Tensor], f64_stats: Dict[str, torch.Tensor],
                         group=None) -> None:
    """In-place all-reduce(sum) of per-gene statistics: all integer arrays travel as one
    int64 buffer, all float64 arrays as one float64 buffer (two collectives in total)."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return
    for stats, dt in ((int_stats, torch.int64), (f64_stats, torch.float64)):
        if not stats:
            continue
        keys = sorted(stats)
        flat = torch.cat([stats[k].reshape(-1).to(dt) for k in keys])
        dist.all_reduce(flat, op=dist.ReduceOp.SUM, group=group)
        off = 0
        for k in keys:
            n = stats[k].numel()
            stats[k].copy_(flat[off:off + n].reshape(stats[k].shape).to(stats[k].dtype))
            off += n


def global_cell_count(n_local: int, device, group=None) -> int:
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return int(n_local)
    t = torch.tensor([n_local], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return int(t[0])


def _need_blocks(n_cols: int, which_moments: int):
    nb = B.rsc_moments_split_blocks(n_cols, which_moments)
    nb = nb if 0 < len(nb) <= 32 else []
    return (C.c_int32 * max(1, len(nb)))(*nb), len(nb)


def preprocess_sharded(pp: "B.Preprocessor", X: "B.Csr", gene_flags: Optional[torch.Tensor],
                       events=None, group=None) -> dict:
    """QC -> all-reduce -> fused pass (raw sums) -> all-reduce -> finalize -> HVG.
    Per-cell outputs describe the local shard; per-gene outputs and the HVG set are global
    and identical on every rank."""
    L, o, p = B.lib(), pp.out, pp.params
    st = torch.cuda.current_stream()
    sp = C.c_void_p(st.cuda_stream)
    cs = X.c_struct()
    G = X.n_cols
    if not hasattr(pp, "_sh"):
        n, nnz = X.n_rows, X.nnz
        pp._sh = dict(
            w0=B._ws(L.rsc_qc_metrics_workspace_bytes(n, G, nnz), X.device),
            w1=B._ws(L.rsc_normalize_log1p_moments_workspace_bytes(n, G, nnz), X.device),
            w2=B._ws(L.rsc_hvg_select_workspace_bytes(G, p.n_bins), X.device),
            splits=(torch.empty(max(1, B.rsc_row_splits_count(n, G)), dtype=torch.int32,
                                device=X.device) if X.sorted_indices else None),
            need=_need_blocks(G, p.which_moments),        # split entries the fused pass reads
            sums=torch.zeros(4, G, dtype=torch.float64, device=X.device),
            n_total=global_cell_count(n, X.device, group))
    sh = pp._sh
    if events:
        events[0].record(st)
    B._check(L.rsc_qc_metrics_splits(C.byref(cs), B._ptr(gene_flags), B._ptr(o["cell_total_i64"]),
                                     B._ptr(o["cell_total_f32"]), B._ptr(o["cell_n_genes"]),
                                     B._ptr(o["cell_flag_total_i64"]), B._ptr(o["cell_flag_pct"]),
                                     B._ptr(o["gene_n_cells"]), B._ptr(o["gene_total_i64"]),
                                     B._ptr(sh["splits"]), C.cast(sh["need"][0], C.c_void_p),
                                     sh["need"][1], B._ptr(sh["w0"]), sh["w0"].numel(), sp))
    allreduce_gene_stats({"n_cells": o["gene_n_cells"], "total": o["gene_total_i64"]}, {}, group)
    if events:
        events[1].record(st)
    B._check(L.rsc_normalize_log1p_moments(
        C.byref(cs), p.target_sum, B._ptr(o["cell_total_i64"]), B._ptr(o["gene_n_cells"]),
        B._ptr(sh["splits"]), p.which_moments, p.ddof, B._ptr(o["mean_log"]), B._ptr(o["var_log"]),
        B._ptr(o["mean_lin"]), B._ptr(o["var_lin"]), B._ptr(sh["sums"]), B._ptr(sh["w1"]),
        sh["w1"].numel(), sp))
    allreduce_gene_stats({}, {"sums": sh["sums"]}, group)
    s = sh["sums"]
    if p.which_moments & B.RSC_MOMENTS_LOG:
        B._check(L.rsc_moments_finalize(G, sh["n_total"], p.ddof, B._ptr(s[0]), B._ptr(s[1]),
                                        B._ptr(o["mean_log"]), B._ptr(o["var_log"]), sp))
    if p.which_moments & B.RSC_MOMENTS_LIN:
        B._check(L.rsc_moments_finalize(G, sh["n_total"], p.ddof, B._ptr(s[2]), B._ptr(s[3]),
                                        B._ptr(o["mean_lin"]), B._ptr(o["var_lin"]), sp))
    if events:
        events[2].record(st)
    hm, hv = (o["mean_lin"], o["var_lin"]) if p.hvg_on_linear else (o["mean_log"], o["var_log"])
    B._check(L.rsc_hvg_select(G, B._ptr(hm), B._ptr(hv), p.n_top, p.n_bins, p.hvg_flags,
                              B._ptr(o["hvg_mean_t"]), B._ptr(o["hvg_disp"]),
                              B._ptr(o["hvg_disp_norm"]), B._ptr(o["hvg_bin"]), B._ptr(o["hvg_mask"]),
                              B._ptr(o["hvg_indices"]), B._ptr(o["hvg_count"]), B._ptr(sh["w2"]),
                              sh["w2"].numel(), sp))
    if events:
        events[3].record(st)
    return o
