#!/usr/bin/env python
"""bench.py — throughput of the whole hot path (QC -> fused normalise+log1p+moments -> HVG)
on BASELINE.json's 1 M-cell configuration, one process per GPU.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A step is one pass of the whole chain over one synthetic matrix resident in HBM.  Prints ONE
JSON line (rank 0).  `value` = nnz/s, device-timed with CUDA events; `e2e` = the same metric
through rsc_preprocess_host with HOST buffers (H2D + D2H inside the timed region);
`roofline` = the dominant kernel (fused pass) against the measured HBM copy rate;
`cpu_baseline` = the CPU oracle on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
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
BYTES_PER_NNZ = {"qc": 8.0, "fused": 12.0, "chain": 20.0}   # SURVEY.md §8(d), DESIGN.md §7
# dram__bytes_read.sum + dram__bytes_write.sum of one fused-pass launch, from the ncu --set full
# capture E in profiles/r01c_cfg3.md; key = (config, which_moments), full-size runs only
NCU_TRAFFIC_BYTES = {(3, 1): 11.979356e9 + 5.863033e9}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number (1-5)")
    ap.add_argument("--cells", type=int, default=None, help="override the row count (debug)")
    ap.add_argument("--which-moments", type=int, default=1,
                    help="moment sets of the fused pass: 1 log scale (north_star's chain, default), "
                         "2 linear scale (scanpy's Seurat input), 3 both")
    ap.add_argument("--no-variants", action="store_true",
                    help="skip the extra timing of the other which-moments settings")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-sample-nnz", type=float, default=2.0e7)
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.index, self.period, self.stop_flag = index, period_s, False
        self.sm, self.reasons, self.max_sm, self.ok = [], 0, None, False
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
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.reasons |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
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
        return {"sm_mhz": float(s[len(s) // 2]), "sm_max_mhz": float(self.max_sm), "reasons": rs,
                "samples": len(s)}


def cpu_oracle_sample(indptr, indices, data, flags, cfg, target_nnz):
    """Time the oracle chain, as it stands, on the first rows of the workload."""
    import numpy as np
    from oracle import oracle_np as O
    ip = indptr.cpu().numpy()
    m = int(np.searchsorted(ip, target_nnz))
    m = max(2, min(m, len(ip) - 1))
    ip = ip[: m + 1]
    k = int(ip[-1])
    ix = indices[:k].cpu().numpy()
    dt = data[:k].cpu().numpy()
    fl = flags.cpu().numpy()
    t0 = time.perf_counter()
    O.preprocess_chain(ip, ix, dt, cfg.n_genes, fl, cfg.target_sum, cfg.n_top, cfg.n_bins)
    sec = time.perf_counter() - t0
    return k / sec, sec, m, k


def run_reference(args):
    """--impl reference: the CPU oracle (the only reference this tier has) on bounded samples."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    from paper_2603_02402_b200 import synth
    cfg = synth.CONFIGS[args.config]
    n_rows = max(64, int(args.cpu_sample_nnz / 1500))
    indptr, indices, data = synth.make_csr(cfg, "cpu", n_cells=n_rows)
    flags = synth.gene_flags(cfg, "cpu")
    times = []
    for i in range(args.warmup + args.steps):
        v, sec, m, k = cpu_oracle_sample(indptr, indices, data, flags, cfg, 1e18)
        if i >= args.warmup:
            times.append(sec)
    nnz = int(indices.numel())
    ms = 1e3 * sum(times) / len(times)
    val = nnz / (ms / 1e3)
    sample = f"first {n_rows} cells of {cfg.name} ({nnz} nnz) per step, full oracle chain"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    import torch.distributed as dist
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

    base = synth.CONFIGS[args.config]
    n_cells = base.n_cells if args.cells is None else args.cells
    # weak scaling: every rank holds its own shard of `n_cells` cells (different seed)
    from dataclasses import replace
    cfg = replace(base, seed=base.seed + 7919 * rank)
    indptr, indices, data = synth.make_csr(cfg, dev, n_cells=n_cells)
    flags = synth.gene_flags(cfg, dev)
    pristine = data.clone()
    X = Csr(indptr, indices, data, cfg.n_genes)
    nnz = X.nnz
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

    for _ in range(max(args.warmup, 3)):
        data.copy_(pristine)
        step_fn(None)
    barrier()

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    launches0 = binding.rsc_kernel_launch_count()
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    for k in range(args.steps):
        data.copy_(pristine)          # restore the raw counts (in-place chain); untimed
        step_fn(evs[k])
    barrier()
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

    # ---- the other moment-set settings of the fused pass, timed the same way (N=1 only)
    variants = None
    if not args.no_variants and world == 1:
        variants = {}
        for wm in (1, 2, 3):
            if wm == args.which_moments:
                continue
            vp = Preprocessor(X.n_rows, X.n_cols, nnz, cfg.target_sum, cfg.n_top, cfg.n_bins, 1,
                              wm, bool(wm & 2), device=dev)
            vevs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(8)]
            for k in range(8):
                data.copy_(pristine)
                vp.run_staged(X, flags, vevs[k] if k >= 3 else None)
            torch.cuda.synchronize()
            tf = [e[1].elapsed_time(e[2]) for e in vevs[3:]]
            tc = [e[0].elapsed_time(e[3]) for e in vevs[3:]]
            variants[f"which_moments={wm}"] = {"fused_ms": sum(tf) / len(tf), "chain_ms": sum(tc) / len(tc),
                                               "chain_nnz_per_s": nnz / (sum(tc) / len(tc) / 1e3)}
            del vp

    # ---- SURVEY 8(f) NEXT-1 on the same matrix: QC-threshold filter + HVG column subsetting
    next1 = None
    if not args.no_variants and world == 1:
        data.copy_(pristine)
        q = binding.rsc_qc_metrics(X, flags)
        out_h = pp.run_staged(X, flags, None)              # leaves the HVG mask of the headline run
        data.copy_(pristine)
        legs = {"filter (min_genes=200, min_cells=3)": binding.rsc_filter_masks(q, min_genes=200, min_cells=3),
                "hvg columns": (None, out_h["hvg_mask"])}
        next1 = {}
        for name, (ck, gk) in legs.items():
            ts, Y = [], None
            for k in range(6):
                del Y
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); Y, g2 = binding.rsc_subset_csr(X, ck, gk); b.record()
                torch.cuda.synchronize()
                if k >= 2:
                    ts.append(a.elapsed_time(b))
            ms = sum(ts) / len(ts)
            byt = 4.0 * nnz + 8.0 * nnz + 8.0 * Y.nnz       # plan reads indices; fill reads both, writes kept
            next1[name] = {"ms": ms, "nnz_out": Y.nnz, "n_rows_out": Y.n_rows, "n_cols_out": g2,
                           "GBps": byt / (ms / 1e3) / 1e9,
                           "note": "plan + size read-back + allocation + fill, CUDA events"}
        # NEXT-3 (first half): dense z-scores of the HVG-subset matrix (Y of the last leg)
        sel = torch.nonzero(out_h["hvg_mask"]).flatten()
        mu, vv = out_h["mean_log"][sel].contiguous(), out_h["var_log"][sel].contiguous()
        ts = []
        for k in range(5):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); Zs = binding.rsc_scale_dense(Y, mu, vv, 10.0, True); b.record()
            torch.cuda.synchronize()
            if k >= 2:
                ts.append(a.elapsed_time(b))
            del Zs
        ms = sum(ts) / len(ts)
        next1["scale (dense, HVG columns, max_value=10)"] = {
            "ms": ms, "out_elements": Y.n_rows * g2,
            "GBps": (4.0 * Y.n_rows * g2 + 8.0 * Y.nnz) / (ms / 1e3) / 1e9,
            "note": "writes n_rows x n_cols float32; reads the subset CSR"}
        del Y, q

    # ---- end to end through the host entry point (rank-local; N=1 only)
    e2e = None
    if not args.no_e2e and world == 1:
        hX = Csr(indptr.cpu().pin_memory(), indices.cpu().pin_memory(), pristine.cpu().pin_memory(),
                 cfg.n_genes)
        hflags = flags.cpu().pin_memory()
        hp = HostPreprocessor(hX.n_rows, hX.n_cols, hX.nnz, cfg.target_sum, cfg.n_top, cfg.n_bins, 1,
                              args.which_moments, hvg_on_linear, device=dev)
        hp.run(hX, hflags); torch.cuda.synchronize()
        ts = []
        for _ in range(max(1, args.e2e_steps)):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record(); hp.run(hX, hflags); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        e2e_ms = sum(ts) / len(ts)
        e2e = {"value": nnz / (e2e_ms / 1e3), "unit": UNIT, "ms_per_step": e2e_ms,
               "h2d_bytes_per_step": hp.h2d_bytes, "d2h_bytes_per_step": hp.d2h_bytes,
               "note": "rsc_preprocess_host: pinned host CSR in, all QC/moment/HVG arrays out; "
                       "x'' stays on the device"}
        del hp, hX

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak()
    avg = lambda v: sum(v) / len(v)      # noqa: E731
    fused_ms, qc_ms, hvg_ms, step_ms = avg(t_fused), avg(t_qc), avg(t_hvg), avg(t_step)
    achieved = BYTES_PER_NNZ["fused"] * nnz / (fused_ms / 1e3) / 1e9
    roofline = {"bound": "hbm", "kernel": "rsc_normalize_log1p_moments (fused pass)",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "peak_source": peak_src,
                "traffic": NCU_TRAFFIC_BYTES.get((args.config, args.which_moments)) if args.cells is None else None,
                "traffic_source": "profiles/r01c_cfg3.md (ncu --set full, bytes per launch)",
                "algorithmic_bytes_per_nnz": BYTES_PER_NNZ["fused"],
                "ms_per_launch": fused_ms, "frac_of_8TBs": achieved / NOMINAL_HBM_GBS}
    stages = {
        "qc": {"ms": qc_ms, "GBps": BYTES_PER_NNZ["qc"] * nnz / (qc_ms / 1e3) / 1e9},
        "fused": {"ms": fused_ms, "GBps": achieved},
        "hvg": {"ms": hvg_ms},
        "chain": {"ms": step_ms, "GBps": BYTES_PER_NNZ["chain"] * nnz / (step_ms / 1e3) / 1e9},
    }
    stages["chain"]["frac_of_8TBs"] = stages["chain"]["GBps"] / NOMINAL_HBM_GBS
    stages["chain"]["frac_of_measured"] = stages["chain"]["GBps"] / peak

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        v, sec, m, k = cpu_oracle_sample(indptr, indices, pristine, flags, cfg, args.cpu_sample_nnz)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": sec,
               "sample": f"first {m} cells of the workload ({k} nnz), full oracle chain once"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": total_ms_max / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": cfg.name if args.cells is None else f"{cfg.name}[:{n_cells}]",
                   "n_cells_per_gpu": X.n_rows, "n_genes": X.n_cols, "nnz_per_gpu": nnz,
                   "target_sum": cfg.target_sum, "n_top": cfg.n_top, "n_bins": cfg.n_bins,
                   "which_moments": args.which_moments,
                   "moments": {1: "log scale (of x'')", 2: "linear scale (of x')", 3: "log + linear"}[args.which_moments & 3],
                   "l2": "inputs (>= 8 B/nnz) larger than L2; data restored from a pristine copy "
                         "between steps (untimed)",
                   "parallelism": "1 GPU" if world == 1 else f"row-sharded x{world} + all-reduce of per-gene sums"},
        "roofline": roofline, "stages": stages, "variants": variants, "next_filter_subset_scale": next1, "cpu_baseline": cpu, "e2e": e2e,
        "gpu_launches": int(launches), "clocks": sampler.summary(),
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
