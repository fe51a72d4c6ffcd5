"""world_size-2 gloo test (CPU) of the row-sharded path's host logic: partial per-gene
statistics from two row shards, one packed all-reduce each, global finalisation — equal to
the single-shard result.  Partials come from the oracle (the kernels need a GPU; their
parity is covered by the -m gpu tests)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import oracle_np as O
from paper_2603_02402_b200 import sharded, synth


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, G = 90, 150
        indptr, indices, data, X = synth.small_nb_csr(n, G, 21, 1.0, empty_rows=(3,), empty_genes=(7,))
        xl = O.log1p(O.normalize_total(indptr, data, 1e4)[0])
        # nnz-balanced shards (config 5's skew is why shards are balanced by nnz, not rows)
        r0, r1 = sharded.nnz_balanced_rows(torch.as_tensor(indptr), world)[rank]
        ip_t, ix_t, dt_t = sharded.shard_csr(torch.as_tensor(indptr), torch.as_tensor(indices),
                                             torch.as_tensor(data), r0, r1)
        ip = ip_t.numpy()
        sl = slice(indptr[r0], indptr[r1])
        assert np.array_equal(ix_t.numpy(), indices[sl]) and np.array_equal(dt_t.numpy(), data[sl])
        q = O.qc_metrics(ip, indices[sl], data[sl], G, None)
        _, _, s1, s2 = O.gene_moments(ip, indices[sl], xl[sl], G) if r1 - r0 > 1 else (0, 0, 0, 0)
        ints = {"n_cells": torch.as_tensor(q["gene_n_cells"].copy()),
                "total": torch.as_tensor(q["gene_total_i64"].copy())}
        f64 = {"sums": torch.as_tensor(np.stack([s1, s2]))}
        sharded.allreduce_gene_stats(ints, f64, exact_in_f64=(rank >= 0))     # one collective for both blocks
        n_total = sharded.global_cell_count(r1 - r0, "cpu")
        assert n_total == n
        assert ints["n_cells"].dtype == torch.int32 and ints["total"].dtype == torch.int64
        qa = O.qc_metrics(indptr, indices, data, G, None)
        assert np.array_equal(ints["n_cells"].numpy(), qa["gene_n_cells"])
        assert np.array_equal(ints["total"].numpy(), qa["gene_total_i64"])
        S1, S2 = f64["sums"][0].numpy(), f64["sums"][1].numpy()
        mean = S1 / n
        var = np.maximum(0.0, (S2 - n * mean * mean) / (n - 1))
        mo, vo, _, _ = O.gene_moments(indptr, indices, xl, G)
        np.testing.assert_allclose(mean, mo, rtol=1e-12)
        np.testing.assert_allclose(var, vo, rtol=1e-9, atol=1e-13)
        h = O.hvg_select(mean, var, 15, 20)
        # every rank ends with the same global selection
        m = torch.as_tensor(h["mask"].astype(np.int64))
        m2 = m.clone(); dist.all_reduce(m2, op=dist.ReduceOp.MAX)
        assert torch.equal(m, m2)
        ret[rank] = "ok"
    finally:
        dist.destroy_process_group()


def test_sharded_allreduce_world2_gloo():
    world = 2
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), ret), nprocs=world, join=True)
    assert dict(ret) == {0: "ok", 1: "ok"}


def test_nnz_balanced_rows():
    rng = np.random.default_rng(0)
    for trial in range(20):
        n = int(rng.integers(1, 400))
        lens = (rng.lognormal(3.0, 1.2, n)).astype(np.int64)          # skewed row lengths
        if trial % 5 == 0:
            lens[rng.integers(0, n, max(1, n // 3))] = 0
        indptr = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        for world in (1, 2, 3, 8):
            parts = sharded.nnz_balanced_rows(torch.as_tensor(indptr), world)
            assert len(parts) == world and parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[k][1] == parts[k + 1][0] for k in range(world - 1))      # contiguous cover
            assert all(r0 <= r1 for r0, r1 in parts)
            nnz = int(indptr[-1])
            longest = int(lens.max()) if n else 0
            for k, (r0, r1) in enumerate(parts):                    # within one row of the ideal cut
                assert abs(int(indptr[r0]) - (nnz * k) // world) <= longest
    # two equal halves
    ip = torch.tensor([0, 5, 10, 15, 20])
    assert sharded.nnz_balanced_rows(ip, 2) == [(0, 2), (2, 4)]


def test_allreduce_is_noop_without_process_group():
    a = {"x": torch.arange(4, dtype=torch.int32)}
    sharded.allreduce_gene_stats(a, {})
    assert a["x"].tolist() == [0, 1, 2, 3]
    assert sharded.global_cell_count(5, "cpu") == 5
