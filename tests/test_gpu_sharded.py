"""The row-sharded chain on the GPU:
world = 1 must reproduce Preprocessor.run_staged bit for bit; world = 2 over NCCL (needs two
GPUs, skipped otherwise) must give every rank the single-GPU per-gene results and HVG set."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2603_02402_b200 import Csr, Preprocessor, sharded, synth

pytestmark = pytest.mark.gpu

GENE_KEYS = ("gene_n_cells", "gene_total_i64", "mean_log", "var_log", "mean_lin", "var_lin",
             "hvg_mean_t", "hvg_disp", "hvg_disp_norm", "hvg_bin", "hvg_mask", "hvg_count")
CELL_KEYS = ("cell_total_i64", "cell_total_f32", "cell_n_genes", "cell_flag_total_i64", "cell_flag_pct")


def _same(a, b):
    return torch.equal(a, b) or (a.is_floating_point() and torch.equal(torch.nan_to_num(a, nan=-7.0),
                                                                       torch.nan_to_num(b, nan=-7.0)))


@pytest.mark.parametrize("which", [1, 3])
def test_sharded_world1_equals_staged(which):
    cfg = synth.scaled(synth.CONFIGS[2], 4000)
    indptr, indices, data = synth.make_csr(cfg, "cuda")
    flags = synth.gene_flags(cfg, "cuda")
    raw = data.clone()
    X = Csr(indptr, indices, data, cfg.n_genes)
    a = Preprocessor(X.n_rows, X.n_cols, X.nnz, cfg.target_sum, 800, cfg.n_bins, 1, which, bool(which & 2))
    ra = {k: v.clone() for k, v in a.run_staged(X, flags).items()}
    xa = X.data.clone()
    X.data.copy_(raw)
    b = Preprocessor(X.n_rows, X.n_cols, X.nnz, cfg.target_sum, 800, cfg.n_bins, 1, which, bool(which & 2))
    rb = sharded.preprocess_sharded(b, X, flags)
    torch.cuda.synchronize()
    assert torch.equal(xa, X.data)
    keys = [k for k in GENE_KEYS + CELL_KEYS if not ((k.endswith("_lin") and not which & 2))]
    for k in keys:
        assert _same(ra[k], rb[k]), k


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _nccl_worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    try:
        cfg = synth.scaled(synth.CONFIGS[5], 6000)           # skewed rows: the nnz-balanced cut matters
        indptr, indices, data = synth.make_csr(cfg, dev)
        flags = synth.gene_flags(cfg, dev)
        raw = data.clone()
        X = Csr(indptr, indices, data, cfg.n_genes)
        one = Preprocessor(X.n_rows, X.n_cols, X.nnz, cfg.target_sum, 900, cfg.n_bins, 1, 3, True, device=dev)
        r1 = {k: v.clone() for k, v in one.run_staged(X, flags).items()}
        x1 = X.data.clone()
        data.copy_(raw)
        r0_, r1_ = sharded.nnz_balanced_rows(indptr, world)[rank]
        ip, ix, dt = sharded.shard_csr(indptr, indices, data, r0_, r1_)
        Xs = Csr(ip, ix.contiguous(), dt.contiguous(), cfg.n_genes)
        pp = Preprocessor(Xs.n_rows, Xs.n_cols, Xs.nnz, cfg.target_sum, 900, cfg.n_bins, 1, 3, True, device=dev)
        rs = sharded.preprocess_sharded(pp, Xs, flags)
        torch.cuda.synchronize()
        ok = torch.equal(Xs.data, x1[int(indptr[r0_]):int(indptr[r1_])])
        for k in ("gene_n_cells", "gene_total_i64", "hvg_mask", "hvg_count", "hvg_bin"):
            ok = ok and torch.equal(rs[k], r1[k])
        for k in ("mean_log", "var_log", "mean_lin", "var_lin"):          # sums are exact integers per shard,
            ok = ok and torch.allclose(rs[k], r1[k], rtol=1e-12, atol=0)  # added in another order across shards
        for k in CELL_KEYS:
            ok = ok and _same(rs[k], r1[k][r0_:r1_])
        ret[rank] = "ok" if ok else "mismatch"
    finally:
        dist.destroy_process_group()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs (NCCL)")
def test_sharded_world2_nccl():
    world = 2
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_nccl_worker, args=(world, _free_port(), ret), nprocs=world, join=True)
    assert dict(ret) == {0: "ok", 1: "ok"}
