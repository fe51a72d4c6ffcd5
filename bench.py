#!/usr/bin/env python
"""bench.py — throughput of the whole hot path (QC -> fused normalise+log1p+moments -> HVG)
on BASELINE.json's 1 M-cell configuration, one process per GPU.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 1..5|all] [--scaling weak|strong]

A step is one pass of the whole chain over one synthetic matrix resident in HBM.  Prints ONE
JSON line (rank 0).  `value` = nnz/s, device-timed with CUDA events; `e2e` = the same metric
through rsc_preprocess_host with HOST buffers (H2D + D2H inside the timed region);
`roofline` = the dominant kernel (fused pass) against the measured HBM copy rate;
`cpu_baseline` = the CPU oracle (C / OpenMP twin, all host cores) on a bounded sample of the same
workload.  The same run also reports (N = 1): the other moment-set settings (`variants`), the
unfused entry points (`unfused`), the SURVEY 8(f) widenings on the same matrix (`next`: filter /
subset / scale / Gram on the tensor cores) and the other BASELINE.json configs (`configs`).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "nnz/s for QC+normalize+log1p+HVG (achieved HBM GB/s in roofline)"
UNIT = "nnz/s"
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json's denominator ("fraction of 8 TB/s")
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent
FALLBACK_BF16_TFLOPS = 1590.0
BYTES_PER_NNZ = {"qc": 8.0, "fused": 12.0, "chain": 20.0}   # SURVEY.md §8(d), DESIGN.md §7
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "traffic.json")   # ncu dram bytes per launch, by kernel / config


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="3",
                    help="headline BASELINE.json config (1-5), or 'all' = config 3 as the headline and "
                         "every other config, config 4 (60 GB) included, in `configs`")
    ap.add_argument("--cells", type=int, default=None, help="override the row count (debug)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank holds its own matrix of the config's size; "
                         "strong = ONE matrix, cut into nnz-balanced row shards")
    ap.add_argument("--which-moments", type=int, default=1,
                    help="moment sets of the fused pass: 1 log scale (north_star's chain, default), "
                         "2 linear scale (scanpy's Seurat input), 3 both")
    ap.add_argument("--no-variants", action="store_true",
                    help="skip variants / unfused / next / other configs (headline only)")
    ap.add_argument("--no-configs", action="store_true", help="skip the other BASELINE.json configs")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-sample-nnz", type=float, default=1.0e8,
                    help="stored entries of the workload's first cells the CPU oracle is timed on")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return (float(d["hbm_gbs"]), float(d.get("bf16_tflops", FALLBACK_BF16_TFLOPS)),
                float(d.get("bf16_tflops_sustained", d.get("bf16_tflops", FALLBACK_BF16_TFLOPS))),
                "measured (MEASURED_PEAKS.json)")
    except Exception:
        return FALLBACK_HBM_GBS, FALLBACK_BF16_TFLOPS, 1400.0, "fallback (B200_PROFILING.md)"


def traffic_of(kernel: str, workload: str):
    """dram read + write bytes of one launch from the tracked ncu capture, or None."""
    try:
        with open(TRAFFIC_FILE) as f:
            d = json.load(f)
        e = d["kernels"][kernel][workload]
        return float(e["dram_bytes_read"]) + float(e["dram_bytes_write"]), d.get("source")
    except Exception:
        return None, None


class ClockSampler(threading.Thread):
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.index, self.period, self.stop_flag = index, period_s, False
        self.recording = False            # samples are kept only while the timed region runs
        self.sm, self.reasons, self.max_sm, self.ok = [], 0, None, False
        self.pw, self.mem = [], []
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_sm = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag:
            try:
                if self.recording:
                    self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                    self.reasons |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                    self.mem.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_MEM))
                    self.pw.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        if not self.ok or not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_sm, "reasons": ["unavailable"]}
        names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap",
                 0x8: "hw_slowdown", 0x10: "sync_boost", 0x20: "sw_thermal_slowdown",
                 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
                 0x100: "display_clock_setting"}
        rs = [v for k, v in names.items() if self.reasons & k and v != "gpu_idle"]
        s = sorted(self.sm)
        return {"sm_mhz": float(s[len(s) // 2]), "sm_mhz_min": float(s[0]), "sm_max_mhz": float(self.max_sm),
                "reasons": rs, "samples": len(s), "power_w_max": max(self.pw) if self.pw else None,
                "mem_mhz_min": min(self.mem) if self.mem else None}


# ------------------------------------------------------------------------------ CPU oracle legs
def _prefix(indptr, indices, data, target_nnz):
    """Host copies of the first cells of the workload holding about target_nnz stored entries."""
    import numpy as np
    ip = indptr.cpu().numpy()
    m = int(np.searchsorted(ip, target_nnz))
    m = max(2, min(m, len(ip) - 1))
    ip = ip[: m + 1].copy()
    k = int(ip[-1])
    return ip, indices[:k].cpu().numpy(), data[:k].cpu().numpy(), m, k


def cpu_oracle_c(ip, ix, dt, flags_np, cfg, repeats=1):
    """The C / OpenMP oracle chain, as it stands, on all host cores: (nnz/s, seconds, threads)."""
    from oracle import build as _ob, oracle_c as OC
    _ob.build()
    OC.lib()
    secs = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        OC.preprocess_chain(ip, ix, dt, cfg.n_genes, flags_np, cfg.target_sum, cfg.n_top, cfg.n_bins)
        secs.append(time.perf_counter() - t0)
    sec = statistics.median(secs)
    return len(ix) / sec, sec, OC.num_threads()


def cpu_oracle_np(ip, ix, dt, flags_np, cfg):
    from oracle import oracle_np as O
    t0 = time.perf_counter()
    O.preprocess_chain(ip, ix, dt, cfg.n_genes, flags_np, cfg.target_sum, cfg.n_top, cfg.n_bins)
    sec = time.perf_counter() - t0
    return len(ix) / sec, sec


def workload_config(cfg, args, n_rows, n_cols, nnz, world, scaling):
    return {"workload": cfg.name if args.cells is None else f"{cfg.name}[:{args.cells}]",
            "n_cells_per_gpu": n_rows, "n_genes": n_cols, "nnz_per_gpu": nnz,
            "target_sum": cfg.target_sum, "n_top": cfg.n_top, "n_bins": cfg.n_bins,
            "which_moments": args.which_moments,
            "moments": {1: "log scale (of x'')", 2: "linear scale (of x')", 3: "log + linear"}[args.which_moments & 3],
            "l2": "inputs (>= 8 B/nnz) larger than L2; data restored from a pristine copy "
                  "between steps (untimed)",
            "parallelism": "1 GPU" if world == 1 else
            f"row-sharded x{world} ({scaling}) + one all-reduce of the per-gene sums"}


def run_reference(args):
    """--impl reference: the CPU oracle (the only reference this tier has; C / OpenMP twin, all host
    cores) on a bounded sample -- the first cells of the SAME matrix the GPU arm times."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    from paper_2603_02402_b200 import synth
    cfgno = 3 if args.config == "all" else int(args.config)
    cfg = synth.CONFIGS[cfgno]
    n_cells = cfg.n_cells if args.cells is None else args.cells
    want_nnz = min(args.cpu_sample_nnz, 5.0e7)
    per_cell = {1: 1500, 2: 2000, 3: 1500, 4: 1500, 5: 3000}[cfgno]
    first = max(64, int(want_nnz / per_cell))
    dev = "cuda" if torch.cuda.is_available() else "cpu"      # same generator as the GPU arm when there is a GPU
    indptr, indices, data = synth.make_csr(cfg, dev, n_cells=n_cells, first_rows=first)
    ip, ix, dt, m, k = _prefix(indptr, indices, data, want_nnz)
    fl = synth.gene_flags(cfg, "cpu").numpy()
    del indptr, indices, data
    times, cores = [], 1
    for i in range(args.warmup + args.steps):
        v, sec, cores = cpu_oracle_c(ip, ix, dt, fl, cfg)
        if i >= args.warmup:
            times.append(sec)
    ms = 1e3 * sum(times) / len(times)
    val = k / (ms / 1e3)
    sample = (f"first {m} cells of {cfg.name} ({k} nnz; generated on {dev}: "
              f"{'the same matrix as the GPU arm' if dev == 'cuda' else 'no GPU here, CPU generator'}) "
              f"per step, full oracle chain (oracle/oracle_c.c, OpenMP)")
    conf = workload_config(cfg, args, n_cells, cfg.n_genes, None, 1, "weak")
    conf["sample"] = sample
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "ms_per_step_median": 1e3 * statistics.median(times), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": conf,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------ GPU legs
def time_chain(torch, pp, X, flags, data, pristine, steps, warmup, step_fn=None):
    """W untimed + K timed passes; returns per-step [qc, fused, hvg, total] ms lists."""
    fn = step_fn if step_fn is not None else (lambda ev: pp.run_staged(X, flags, ev))
    for _ in range(warmup):
        data.copy_(pristine)
        fn(None)
    torch.cuda.synchronize()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
    for k in range(steps):
        data.copy_(pristine)          # restore the raw counts (in-place chain); untimed
        fn(evs[k])
    torch.cuda.synchronize()
    return {"qc": [e[0].elapsed_time(e[1]) for e in evs], "fused": [e[1].elapsed_time(e[2]) for e in evs],
            "hvg": [e[2].elapsed_time(e[3]) for e in evs], "step": [e[0].elapsed_time(e[3]) for e in evs]}


def timed(torch, fn, reps=5, warm=2, before=None):
    ts, r = [], None
    for k in range(reps + warm):
        if before is not None:
            before()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); r = fn(); b.record()
        torch.cuda.synchronize()
        if k >= warm:
            ts.append(a.elapsed_time(b))
    return statistics.median(ts), r


def other_config(torch, synth, binding, Csr, Preprocessor, cfgno, dev, peak):
    """Chain timing of another BASELINE.json config (headline settings: log-scale set)."""
    cfg = synth.CONFIGS[cfgno]
    indptr, indices, data = synth.make_csr(cfg, dev)
    flags = synth.gene_flags(cfg, dev)
    pristine = data.clone()
    X = Csr(indptr, indices, data, cfg.n_genes)
    pp = Preprocessor(X.n_rows, X.n_cols, X.nnz, cfg.target_sum, cfg.n_top, cfg.n_bins, 1, 1, False, device=dev)
    t = time_chain(torch, pp, X, flags, data, pristine, 10, 3)
    ms = statistics.median(t["step"])
    out = {"n_cells": X.n_rows, "n_genes": X.n_cols, "nnz": X.nnz, "chain_ms": ms,
           "qc_ms": statistics.median(t["qc"]), "fused_ms": statistics.median(t["fused"]),
           "hvg_ms": statistics.median(t["hvg"]), "nnz_per_s": X.nnz / (ms / 1e3),
           "chain_GBps": BYTES_PER_NNZ["chain"] * X.nnz / (ms / 1e3) / 1e9}
    out["frac_of_8TBs"] = out["chain_GBps"] / NOMINAL_HBM_GBS
    out["frac_of_measured"] = out["chain_GBps"] / peak
    if cfgno == 1:
        # launch-bound (the matrix fits L2): the same chain replayed from one CUDA graph
        try:
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                pp.run_staged(X, flags, None, stream=st)
                st.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=st):
                    pp.run_staged(X, flags, None, stream=st)
            gms, _ = timed(torch, lambda: g.replay(), reps=10, warm=3, before=lambda: data.copy_(pristine))
            out["chain_ms_cuda_graph"] = gms
        except Exception as e:                                # noqa: BLE001
            out["chain_ms_cuda_graph"] = None
            out["cuda_graph_error"] = str(e)[:200]
    del pp, X, indptr, indices, data, pristine
    torch.cuda.empty_cache()
    return cfg.name, out


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    import torch.distributed as dist
    from dataclasses import replace
    from paper_2603_02402_b200 import Csr, HostPreprocessor, Preprocessor, synth
    from paper_2603_02402_b200 import binding, build as _build

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    _build.build()
    binding.lib()

    cfgno = 3 if args.config == "all" else int(args.config)
    base = synth.CONFIGS[cfgno]
    n_cells = base.n_cells if args.cells is None else args.cells
    scaling = args.scaling if world > 1 else "weak"
    if world > 1 and scaling == "strong":
        # ONE matrix (the config's), cut into nnz-balanced row shards; every rank draws the same
        # matrix from the same seed and keeps its own rows (no host round trip)
        from paper_2603_02402_b200 import sharded
        cfg = base
        ip_all, ix_all, dt_all = synth.make_csr(cfg, dev, n_cells=n_cells)
        r0, r1 = sharded.nnz_balanced_rows(ip_all, world)[rank]
        p0, p1 = int(ip_all[r0]), int(ip_all[r1])
        indptr = (ip_all[r0:r1 + 1] - p0).contiguous()
        indices, data = ix_all[p0:p1].clone(), dt_all[p0:p1].clone()
        del ip_all, ix_all, dt_all
        torch.cuda.empty_cache()
    else:
        # weak scaling: every rank holds its own matrix of `n_cells` cells (different seed)
        cfg = replace(base, seed=base.seed + 7919 * rank)
        indptr, indices, data = synth.make_csr(cfg, dev, n_cells=n_cells)
    flags = synth.gene_flags(cfg, dev)
    pristine = data.clone()
    X = Csr(indptr, indices, data, cfg.n_genes)
    nnz = X.nnz
    n_rows_local = X.n_rows
    hvg_on_linear = bool(args.which_moments & 2)
    pp = Preprocessor(X.n_rows, X.n_cols, nnz, cfg.target_sum, cfg.n_top, cfg.n_bins, 1,
                      args.which_moments, hvg_on_linear, device=dev)

    if world > 1:
        from paper_2603_02402_b200 import sharded
        step_fn = lambda ev: sharded.preprocess_sharded(pp, X, flags, ev)   # noqa: E731
    else:
        step_fn = lambda ev: pp.run_staged(X, flags, ev)                    # noqa: E731

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # everything slow on the host (event creation, NVML initialisation, the sampler thread) happens
    # BEFORE the warm-up, so that the GPU does not idle -- and drop its clocks -- between the last
    # warm-up step and the first timed one
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        data.copy_(pristine)
        step_fn(None)
    barrier()
    launches0 = binding.rsc_kernel_launch_count()
    sampler.recording = True
    for k in range(args.steps):
        data.copy_(pristine)          # restore the raw counts (in-place chain); untimed
        step_fn(evs[k])
    barrier()
    sampler.recording = False
    sampler.stop_flag = True
    sampler.join()
    launches = binding.rsc_kernel_launch_count() - launches0

    t_step = [e[0].elapsed_time(e[3]) for e in evs]
    t_qc = [e[0].elapsed_time(e[1]) for e in evs]
    t_fused = [e[1].elapsed_time(e[2]) for e in evs]
    t_hvg = [e[2].elapsed_time(e[3]) for e in evs]
    total_ms = sum(t_step)
    tt = torch.tensor([total_ms, float(nnz)], dtype=torch.float64, device=dev)
    if world > 1:
        tmax = tt.clone(); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        tsum = tt.clone(); dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
        total_ms_max, nnz_all = float(tmax[0]), float(tsum[1])
    else:
        total_ms_max, nnz_all = total_ms, float(nnz)
    value = nnz_all * args.steps / (total_ms_max / 1e3)
    peak, tf_burst, tf_sust, peak_src = measured_peaks()
    extras = (not args.no_variants) and world == 1

    # ---- the other moment-set settings of the fused pass, timed the same way (N=1 only)
    variants = None
    if extras:
        variants = {}
        for wm in (1, 2, 3):
            if wm == args.which_moments:
                continue
            vp = Preprocessor(X.n_rows, X.n_cols, nnz, cfg.target_sum, cfg.n_top, cfg.n_bins, 1,
                              wm, bool(wm & 2), device=dev)
            t = time_chain(torch, vp, X, flags, data, pristine, 5, 3)
            variants[f"which_moments={wm}"] = {"fused_ms": statistics.median(t["fused"]),
                                               "chain_ms": statistics.median(t["step"]),
                                               "chain_nnz_per_s": nnz / (statistics.median(t["step"]) / 1e3)}
            del vp
        # the one-pass chain (csrc/single.cu, option "single_pass"): QC folded into the fused pass by
        # pairs of CTAs; 12 B / nnz of DRAM traffic, but more instructions than the two passes together
        if args.which_moments == 1 and cfg.n_genes <= 32768:
            sp = Preprocessor(X.n_rows, X.n_cols, nnz, cfg.target_sum, cfg.n_top, cfg.n_bins, 1, 1, False, device=dev)
            binding.rsc_set_option("single_pass", 1)
            try:
                ms_sp, _ = timed(torch, lambda: sp.run(X, flags), reps=5, warm=2,
                                 before=lambda: data.copy_(pristine))
            finally:
                binding.rsc_set_option("single_pass", 0)
            variants["single_pass"] = {"chain_ms": ms_sp, "chain_nnz_per_s": nnz / (ms_sp / 1e3),
                                       "dram_bytes_per_nnz": 12.0,
                                       "note": "rsc_preprocess with option single_pass=1 (not the default)"}
            del sp

    # ---- the unfused entry points, 8 B / nnz each
    unfused = None
    if extras:
        data.copy_(pristine)
        q = binding.rsc_qc_metrics(X, flags)
        restore = lambda: data.copy_(pristine)                               # noqa: E731
        ms_n, _ = timed(torch, lambda: binding.rsc_normalize_total(X, cfg.target_sum, q["cell_total_i64"]),
                        before=restore)
        ms_l, _ = timed(torch, lambda: binding.rsc_log1p(X), before=restore)
        data.copy_(pristine)
        binding.rsc_normalize_total(X, cfg.target_sum, q["cell_total_i64"]); binding.rsc_log1p(X)
        ms_m, _ = timed(torch, lambda: binding.rsc_gene_moments(X, 0, 1))
        unfused = {}
        for name, ms in (("rsc_normalize_total", ms_n), ("rsc_log1p", ms_l), ("rsc_gene_moments", ms_m)):
            gb = 8.0 * nnz / (ms / 1e3) / 1e9
            unfused[name] = {"ms": ms, "GBps": gb, "frac_of_measured": gb / peak, "bytes_per_nnz": 8.0}
        unfused["note"] = ("separate C-ABI calls on the same matrix; rsc_gene_moments on the log-normalised "
                           "values (transform 0, on-chip integer accumulators)")
        del q

    # ---- SURVEY 8(f) on the same matrix: QC-threshold filter, HVG column subset, scale, Gram
    nxt = None
    if extras:
        data.copy_(pristine)
        q = binding.rsc_qc_metrics(X, flags)
        out_h = pp.run_staged(X, flags, None)              # leaves x'' in X and the HVG mask of the headline run
        legs = {"filter (min_genes=200, min_cells=3)": binding.rsc_filter_masks(q, min_genes=200, min_cells=3),
                "hvg columns": (None, out_h["hvg_mask"])}
        nxt = {}
        Y, g2 = None, 0
        for name, (ck, gk) in legs.items():
            del Y
            ms, (Y, g2) = timed(torch, lambda: binding.rsc_subset_csr(X, ck, gk), reps=4, warm=2)
            # plan reads indices (not when every column is kept: a pure row filter); fill reads both, writes kept
            byt = (0.0 if g2 == X.n_cols else 4.0 * nnz) + 8.0 * nnz + 8.0 * Y.nnz
            nxt[name] = {"ms": ms, "nnz_out": Y.nnz, "n_rows_out": Y.n_rows, "n_cols_out": g2,
                         "GBps": byt / (ms / 1e3) / 1e9,
                         "note": "plan + size read-back + allocation + fill, CUDA events"}
        # NEXT-3, first half: dense z-scores of the HVG-subset matrix (Y of the last leg)
        sel = torch.nonzero(out_h["hvg_mask"]).flatten()
        mu, vv = out_h["mean_log"][sel].contiguous(), out_h["var_log"][sel].contiguous()
        ms, Zs = timed(torch, lambda: binding.rsc_scale_dense(Y, mu, vv, 10.0, True), reps=3, warm=2)
        del Zs
        nxt["scale (dense, HVG columns, max_value=10)"] = {
            "ms": ms, "out_elements": Y.n_rows * g2,
            "GBps": (4.0 * Y.n_rows * g2 + 8.0 * Y.nnz) / (ms / 1e3) / 1e9,
            "note": "writes n_rows x n_cols float32; reads the subset CSR"}
        # NEXT-3, second half: Gram / covariance of the HVG-subset matrix on the tensor cores
        ms, Gc = timed(torch, lambda: binding.rsc_gram_cov(Y), reps=3, warm=2)
        del Gc
        fl = 3.0 * Y.n_rows * float(g2) * float(g2)         # 3 fp16 products x upper triangle (2 n p^2 / 2)
        nxt["gram_cov (HVG columns, tcgen05)"] = {
            "ms": ms, "n": Y.n_rows, "p": g2, "TFLOPs": fl / (ms / 1e3) / 1e12,
            "roofline": {"bound": "tensor", "achieved": fl / (ms / 1e3) / 1e12, "peak": tf_burst, "unit": "TFLOP/s",
                         "frac": fl / (ms / 1e3) / 1e12 / tf_burst,
                         "peak_source": peak_src + " bf16_tflops (burst); fp16 = bf16 rate (guide's nominal ratio 1)",
                         "flops": "3 n p^2: hi*hi + hi*lo + lo*hi on the upper triangle; tile padding not counted"},
            "note": "whole rsc_gram_cov call: exact mean (moments pass), pack to fp16 hi/lo planes, MMA, finalize"}
        # log-scale moments of the HVG columns only: what `scale` needs when the chain ran with the
        # linear-scale set alone (the scanpy order: HVG from x', scale on the subset) -- the cheap
        # alternative to which_moments = 3
        ms, _mm = timed(torch, lambda: binding.rsc_gene_moments(Y, 0, 1), reps=3, warm=2)
        nxt["gene_moments (HVG columns, log scale)"] = {
            "ms": ms, "GBps": 8.0 * Y.nnz / (ms / 1e3) / 1e9,
            "note": "with variants.which_moments=2 this replaces the two-set fused pass: chain(2) + subset + this"}
        if variants is not None and "which_moments=2" in variants:
            nxt["gene_moments (HVG columns, log scale)"]["two_set_workflow_ms"] = \
                variants["which_moments=2"]["chain_ms"] + ms
        # the projection of L95 on 50 loadings (orthonormal random V: the eigensolver is a library call)
        Vq = torch.linalg.qr(torch.randn(g2, 50, dtype=torch.float64, device=dev))[0].contiguous()
        mu64 = out_h["mean_log"][sel].contiguous()
        ms, Zp = timed(torch, lambda: binding.rsc_pca_transform(Y, Vq, mu64), reps=3, warm=2)
        del Zp, Vq
        nxt["pca_transform (HVG columns, 50 components)"] = {
            "ms": ms, "GBps_L2_table_reads": 200.0 * Y.nnz / (ms / 1e3) / 1e9,
            "note": "Z = XV - 1 mu^T V; a 200-byte row of the float32 V table per stored entry (L2 / L1), fp64 accumulation"}
        del Y, q

    # ---- end to end through the host entry point (rank-local; N=1 only)
    e2e = None
    e2e_rt = None
    have_matrix = True
    if not args.no_e2e and world == 1 and have_matrix:
        hX = Csr(indptr.cpu().pin_memory(), indices.cpu().pin_memory(), pristine.cpu().pin_memory(),
                 cfg.n_genes)
        hflags = flags.cpu().pin_memory()
        for roundtrip in (False, True):
            hp = HostPreprocessor(hX.n_rows, hX.n_cols, hX.nnz, cfg.target_sum, cfg.n_top, cfg.n_bins, 1,
                                  args.which_moments, hvg_on_linear, device=dev, copy_back_data=roundtrip)
            hp.run(hX, hflags); torch.cuda.synchronize()
            ts = []
            for _ in range(max(1, args.e2e_steps)):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                a.record(); hp.run(hX, hflags); b.record()
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
            ms = statistics.median(ts)
            r = {"value": nnz / (ms / 1e3), "unit": UNIT, "ms_per_step": ms,
                 "h2d_bytes_per_step": hp.h2d_bytes, "d2h_bytes_per_step": hp.d2h_bytes,
                 "note": "rsc_preprocess_host: pinned host CSR in (row chunks: H2D of chunk k+1 and D2H of chunk k-1 "
                         "beside the kernels of chunk k), all QC/moment/HVG arrays out; " +
                         ("the log-normalised x'' copied back to the host as well" if roundtrip else
                          "x'' stays on the device")}
            if roundtrip:
                e2e_rt = r
            else:
                e2e = r
            del hp
        del hX

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    fused_ms, qc_ms, hvg_ms = statistics.median(t_fused), statistics.median(t_qc), statistics.median(t_hvg)
    step_ms = total_ms / args.steps
    achieved = BYTES_PER_NNZ["fused"] * nnz / (fused_ms / 1e3) / 1e9
    wl = cfg.name if args.cells is None else f"{cfg.name}[:{n_cells}]"
    kern = {1: "fused_stream_kernel<1,0>", 2: "fused_stream_kernel<0,1>", 3: "fused_stream_kernel<1,1>"}[args.which_moments & 3]
    traffic, tsrc = traffic_of(kern, wl)
    roofline = {"bound": "hbm", "kernel": "rsc_normalize_log1p_moments (fused pass)",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "peak_source": peak_src + " hbm_gbs",
                "traffic": traffic, "traffic_source": tsrc,
                "algorithmic_bytes_per_nnz": BYTES_PER_NNZ["fused"],
                "ms_per_launch": fused_ms, "frac_of_8TBs": achieved / NOMINAL_HBM_GBS}
    # this board's own copy rate, measured the way MEASURED_PEAKS.json's was (context for the box-to-box
    # spread of the fused pass; `peak` stays the driver's number)
    try:
        ca = torch.empty(1 << 30, dtype=torch.bfloat16, device=dev)
        cb = torch.empty_like(ca)
        best = None
        for _ in range(6):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); cb.copy_(ca); e1.record(); torch.cuda.synchronize()
            ms_c = e0.elapsed_time(e1)
            best = ms_c if best is None or ms_c < best else best
        roofline["copy_rate_this_board_GBps"] = 2 * ca.numel() * 2 / (best / 1e3) / 1e9
        roofline["frac_of_this_board"] = achieved / roofline["copy_rate_this_board_GBps"]
        del ca, cb
    except Exception:                                          # noqa: BLE001
        roofline["copy_rate_this_board_GBps"] = None
    qc_gb = BYTES_PER_NNZ["qc"] * nnz / (qc_ms / 1e3) / 1e9
    stages = {
        "qc": {"ms": qc_ms, "GBps": qc_gb, "frac_of_measured": qc_gb / peak},
        "fused": {"ms": fused_ms, "GBps": achieved, "frac_of_measured": achieved / peak},
        "hvg": {"ms": hvg_ms},
        "chain": {"ms": step_ms, "ms_median": statistics.median(t_step),
                  "GBps": BYTES_PER_NNZ["chain"] * nnz / (step_ms / 1e3) / 1e9},
    }
    stages["chain"]["frac_of_8TBs"] = stages["chain"]["GBps"] / NOMINAL_HBM_GBS
    stages["chain"]["frac_of_measured"] = stages["chain"]["GBps"] / peak

    cpu = None
    if not args.no_cpu_baseline and world == 1 and have_matrix:
        ip, ix, dt, m, k = _prefix(indptr, indices, pristine, args.cpu_sample_nnz)
        fl = flags.cpu().numpy()
        try:
            v, sec, cores = cpu_oracle_c(ip, ix, dt, fl, cfg, repeats=3)
            cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": sec,
                   "sample": f"first {m} cells of the workload ({k} nnz), full oracle chain "
                             f"(oracle/oracle_c.c, OpenMP, all host cores), median of 3"}
        except Exception as e:                                # noqa: BLE001
            cpu = {"error": str(e)[:200]}
        ip2, ix2, dt2, m2, k2 = _prefix(indptr, indices, pristine, 2.0e7)
        v1, s1 = cpu_oracle_np(ip2, ix2, dt2, fl, cfg)
        cpu["numpy_1_core"] = {"value": v1, "unit": UNIT, "cores": 1, "seconds": s1,
                               "sample": f"first {m2} cells ({k2} nnz), oracle/oracle_np.py once"}
        cpu["context"] = ("a reported baseline, not the target; the paper quotes ~70x for its preprocessing "
                          "stage on a B200 against a 32-core Threadripper Pro 7975WX (PAPER.md:L49, L145)")

    # ---- the other BASELINE.json configs, same chain, same run
    configs = None
    if extras and args.cells is None and not args.no_configs:
        configs = {}
        others = [c for c in (1, 2, 5, 4) if c != cfgno]
        if args.config != "all":
            others = [c for c in others if c != 4]           # 60 GB + pristine copy: on request only
        keep = (indptr, indices, data, pristine, X)
        for c in others:
            if c == 4:                                        # needs ~100 GB: release the headline matrix first
                del keep, indptr, indices, data, pristine, X
                torch.cuda.empty_cache()
            try:
                name, res = other_config(torch, synth, binding, Csr, Preprocessor, c, dev, peak)
                configs[name] = res
            except Exception as e:                            # noqa: BLE001
                configs[f"cfg{c}"] = {"error": str(e)[:300]}
                torch.cuda.empty_cache()

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": total_ms_max / args.steps,
        "ms_per_step_median": statistics.median(t_step),
        "ms_per_step_min_max": [min(t_step), max(t_step)],
        "higher_is_better": True, "scaling": scaling, "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": workload_config(cfg, args, n_rows_local, cfg.n_genes, nnz, world, scaling),
        "roofline": roofline, "stages": stages, "variants": variants, "unfused": unfused,
        "next": nxt, "configs": configs, "cpu_baseline": cpu, "e2e": e2e, "e2e_roundtrip": e2e_rt,
        "gpu_launches": int(launches), "clocks": sampler.summary(),
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
