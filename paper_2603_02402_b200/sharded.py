"""Row-sharded multi-GPU chain: one process per GPU, each holding a shard of the cells.

The paper scales out by partitioning the matrix "into chunks along the cell axis ... distributed
evenly across available devices" (Dask).  Here the same partitioning runs as one
process per GPU over `torch.distributed`: per-cell outputs, normalisation and log1p are
independent per row; the per-gene integer counts / totals and the double-precision sums S1, S2
need ONE exchange -- an all-reduce(sum) of one contiguous per-gene block (<= 36 k genes x 6 values
~ 1.7 MB, latency-bound on NVLink) AFTER the fused pass (the fused pass balances its gene groups
with the LOCAL counts, which serve as well as the global ones; nothing waits on a collective
between the two streaming passes) -- after which every rank finalises the moments with the global
cell count and runs the identical HVG selection.  Shards are cut by stored entries, not by rows
(`nnz_balanced_rows`; BASELINE.json config 5's row lengths span 50 .. 25 000).

`allreduce_gene_stats`, `nnz_balanced_rows` and `shard_csr` are device-agnostic, so the host-side
logic is covered by world_size-2 gloo tests on CPU; the kernels are the same single-GPU C-ABI calls.
"""
from __future__ import annotations

import ctypes as C
from typing import Dict, Optional

import torch
import torch.distributed as dist

from . import binding as B


def nnz_balanced_rows(indptr: torch.Tensor, world: int):
    """Cut the rows into `world` contiguous shards holding (nearly) equal numbers of stored
    entries: shard k = rows [r_k, r_{k+1}) with r_k = the first row whose offset reaches
    k * nnz / world.  Returns [(r0, r1)] * world (empty shards possible when world > rows)."""
    ip = torch.as_tensor(indptr)
    n = ip.numel() - 1
    nnz = int(ip[-1])
    targets = torch.tensor([(nnz * k) // world for k in range(1, world)], dtype=ip.dtype, device=ip.device)
    cuts = torch.searchsorted(ip[:-1].contiguous(), targets, right=False).tolist() if world > 1 else []
    bounds = [0] + [min(max(int(c), 0), n) for c in cuts] + [n]
    for k in range(1, len(bounds)):
        bounds[k] = max(bounds[k], bounds[k - 1])
    return [(bounds[k], bounds[k + 1]) for k in range(world)]


def shard_csr(indptr: torch.Tensor, indices: torch.Tensor, data: torch.Tensor, r0: int, r1: int):
    """Rows [r0, r1) as a CSR of their own (offsets rebased; indices / data are views)."""
    p0, p1 = int(indptr[r0]), int(indptr[r1])
    return (indptr[r0:r1 + 1] - p0).contiguous(), indices[p0:p1], data[p0:p1]


def allreduce_gene_stats(int_stats: Dict[str, torch.Tensor], f64_stats: Dict[str, torch.Tensor],
                         group=None, exact_in_f64: bool = False) -> None:
    """In-place all-reduce(sum) of per-gene statistics.  All integer arrays travel as one int64
    buffer and all float64 arrays as one float64 buffer (two collectives, back to back); with
    exact_in_f64 (the caller guarantees every integer total stays below 2^53) the integers ride
    in the float64 buffer and ONE collective moves everything."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return
    if exact_in_f64 and int_stats and f64_stats:
        ki, kf = sorted(int_stats), sorted(f64_stats)
        flat = torch.cat([int_stats[k].reshape(-1).to(torch.float64) for k in ki] +
                         [f64_stats[k].reshape(-1) for k in kf])
        dist.all_reduce(flat, op=dist.ReduceOp.SUM, group=group)
        off = 0
        for stats, keys in ((int_stats, ki), (f64_stats, kf)):
            for k in keys:
                n = stats[k].numel()
                stats[k].copy_(flat[off:off + n].reshape(stats[k].shape).to(stats[k].dtype))
                off += n
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
    """QC -> fused pass (raw sums) -> ONE all-reduce of the per-gene block -> finalize -> HVG.
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
    if events:
        events[1].record(st)
    B._check(L.rsc_normalize_log1p_moments(
        C.byref(cs), p.target_sum, B._ptr(o["cell_total_i64"]), B._ptr(o["gene_n_cells"]),
        B._ptr(sh["splits"]), p.which_moments, p.ddof, B._ptr(o["mean_log"]), B._ptr(o["var_log"]),
        B._ptr(o["mean_lin"]), B._ptr(o["var_lin"]), B._ptr(sh["sums"]), B._ptr(sh["w1"]),
        sh["w1"].numel(), sp))
    # counts < 2^31 and totals < n_total * 2^24 (QC precondition) are exact in float64 below 2^29 cells
    allreduce_gene_stats({"n_cells": o["gene_n_cells"], "total": o["gene_total_i64"]}, {"sums": sh["sums"]},
                         group, exact_in_f64=sh["n_total"] < (1 << 29))
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
