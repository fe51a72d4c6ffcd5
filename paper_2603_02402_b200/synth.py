"""Seeded synthetic CSR count matrices (input source only).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's arithmetic: it only draws negative-binomial count
matrices with the shape of single-cell UMI data and returns them as CSR arrays
(float32 data, int32 indices, int64 indptr).  It imports neither ``oracle`` nor
the CUDA binding.

The paper measured on the 10x Genomics 1.3 M mouse-brain data set and on
Tahoe-100M ("Performance and reproducibility" /
"Benchmarking"); neither is available, so BASELINE.json's five seeded
negative-binomial configurations stand in for them (recipe in DESIGN.md §4):

* gene abundance  g_j ~ LogNormal(-1.5, 1.5)
* cell size factor s_c ~ LogNormal(0, sigma_s)   (0.5; config 5: 1.2)
* count x_ij ~ NB(mean = depth * s_c * g_j, theta = 2), zeros dropped,
  columns ascending inside a row
* config 5 adds 200 "housekeeping" genes with mean 20 in every cell
* ``depth`` calibrates nnz/cell to the figure BASELINE.json states.

theta = 2 makes NB the sum of two geometric variables with success
probability q = 2/(2+mu); each is drawn by exact inversion
floor(ln u / ln(1-q)).  Large configs are drawn on the GPU with torch's
Philox generator in fixed-size row chunks (the chunk size is part of the
recipe: it fixes the order in which random numbers are consumed).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace
from typing import Optional, Tuple

import numpy as np
import torch

__all__ = ["Config", "CONFIGS", "make_csr", "small_nb_csr", "gene_flags"]


@dataclass(frozen=True)
class Config:
    name: str
    n_cells: int
    n_genes: int
    depth: float          # calibrated so that nnz/cell matches BASELINE.json
    sigma_s: float        # sd of log size factor
    n_flagged: int        # first n_flagged genes carry the QC flag ("mt")
    target_sum: float
    n_top: int
    seed: int
    n_bins: int = 20
    n_housekeeping: int = 0
    housekeeping_mu: float = 20.0


# BASELINE.json `configs`, in order.  Depths: SURVEY.md §8(d) calibration.
CONFIGS = {
    1: Config("cfg1_5k_x_18k", 5_000, 18_000, 0.158, 0.5, 13, 1e4, 2000, 0),
    2: Config("cfg2_100k_x_30k", 100_000, 30_000, 0.122, 0.5, 37, 1e4, 2000, 1),
    3: Config("cfg3_1M_x_30k", 1_000_000, 30_000, 0.084, 0.5, 37, 1e4, 4000, 2),
    4: Config("cfg4_5M_x_30k", 5_000_000, 30_000, 0.084, 0.5, 37, 1e4, 2000, 3),
    5: Config("cfg5_skew_500k_x_36k", 500_000, 36_000, 0.10, 1.2, 37, 1e6, 3000, 4,
              n_housekeeping=200),
}

# rows per generation chunk: chunk * n_genes <= 2**26 candidate pairs
_CHUNK_PAIRS = 1 << 26


def gene_flags(cfg: Config, device="cpu") -> torch.Tensor:
    """uint8[n_genes]; the first ``n_flagged`` genes are flagged."""
    f = torch.zeros(cfg.n_genes, dtype=torch.uint8, device=device)
    f[: cfg.n_flagged] = 1
    return f


def _chunk_counts(mu: torch.Tensor, gen: torch.Generator) -> torch.Tensor:
    """NB(mean=mu, theta=2) draws as float32, same shape as ``mu``."""
    # ln(1-q) with q = 2/(2+mu):  1-q = mu/(2+mu)
    log1mq = torch.log(mu) - torch.log(mu + 2.0)
    out = None
    for _ in range(2):
        u = torch.rand(mu.shape, generator=gen, device=mu.device, dtype=torch.float32)
        u = 1.0 - u                      # (0, 1]
        k = torch.floor(torch.log(u) / log1mq)
        out = k if out is None else out + k
    return out


def make_csr(cfg: Config, device="cpu", n_cells: Optional[int] = None, first_rows: Optional[int] = None
             ) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """Draw the configuration's matrix on ``device``.

    Returns (indptr int64[n+1], indices int32[nnz], data float32[nnz]).
    ``n_cells`` overrides the row count (used for bounded samples of a
    workload; the gene parameters stay those of the full configuration).
    ``first_rows`` draws only the first rows OF THE n-CELL MATRIX (whole generation chunks, so
    at least that many rows come back): the same random numbers in the same order, i.e. a true
    prefix of the full matrix at a fraction of the cost.
    """
    n = cfg.n_cells if n_cells is None else int(n_cells)
    G = cfg.n_genes
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(cfg.seed)

    g = torch.exp(-1.5 + 1.5 * torch.randn(G, generator=gen, device=dev))
    hk_mask = torch.zeros(G, dtype=torch.bool, device=dev)
    if cfg.n_housekeeping:
        perm = torch.randperm(G, generator=gen, device=dev)[: cfg.n_housekeeping]
        hk_mask[perm] = True
    s = torch.exp(cfg.sigma_s * torch.randn(n, generator=gen, device=dev))

    rows_per_chunk = max(1, _CHUNK_PAIRS // G)
    # capacity from the expected nnz of a row sample: P(x>0) = 1 - q^2
    ns = min(n, 2048)
    mu_s = cfg.depth * s[:ns, None] * g[None, :]
    if cfg.n_housekeeping:
        mu_s = torch.where(hk_mask[None, :], torch.full_like(mu_s, cfg.housekeeping_mu), mu_s)
    p_nz = 1.0 - (2.0 / (2.0 + mu_s)) ** 2
    per_row = float(p_nz.sum(dim=1).mean())
    del mu_s, p_nz
    cap = int(per_row * n * 1.05) + 4 * rows_per_chunk + 1024
    indices = torch.empty(cap, dtype=torch.int32, device=dev)
    data = torch.empty(cap, dtype=torch.float32, device=dev)
    row_nnz = torch.empty(n, dtype=torch.int64, device=dev)

    pos = 0
    n_draw = n if first_rows is None else min(n, -(-int(first_rows) // rows_per_chunk) * rows_per_chunk)
    for r0 in range(0, n_draw, rows_per_chunk):
        r1 = min(n, r0 + rows_per_chunk)
        mu = cfg.depth * s[r0:r1, None] * g[None, :]
        if cfg.n_housekeeping:
            mu = torch.where(hk_mask[None, :], torch.full_like(mu, cfg.housekeeping_mu), mu)
        x = _chunk_counts(mu, gen)
        del mu
        nz = x > 0
        row_nnz[r0:r1] = nz.sum(dim=1)
        rc = torch.nonzero(nz)             # row-major => columns ascending per row
        k = rc.shape[0]
        if pos + k > cap:
            raise RuntimeError("synth.make_csr: capacity estimate exceeded")
        indices[pos:pos + k] = rc[:, 1].to(torch.int32)
        data[pos:pos + k] = x[nz]
        pos += k
        del x, nz, rc
    indptr = torch.zeros(n_draw + 1, dtype=torch.int64, device=dev)
    torch.cumsum(row_nnz[:n_draw], dim=0, out=indptr[1:])
    return indptr, indices[:pos], data[:pos]


def small_nb_csr(n: int, G: int, seed: int, depth: float = 1.0, sigma_s: float = 0.5,
                 empty_rows=(), empty_genes=()):
    """Tiny NumPy matrices for the CPU tests (numpy.random negative_binomial).

    Returns (indptr int64, indices int32, data float32, dense float64[n, G]).
    ``empty_rows`` / ``empty_genes`` are zeroed to exercise the degenerate cases.
    """
    rng = np.random.default_rng(seed)
    g = np.exp(-1.5 + 1.5 * rng.standard_normal(G))
    s = np.exp(sigma_s * rng.standard_normal(n))
    mu = depth * s[:, None] * g[None, :]
    x = rng.negative_binomial(2, 2.0 / (2.0 + mu)).astype(np.float64)
    for r in empty_rows:
        x[r, :] = 0
    for c in empty_genes:
        x[:, c] = 0
    indptr = np.zeros(n + 1, dtype=np.int64)
    nzr, nzc = np.nonzero(x)
    np.cumsum(np.bincount(nzr, minlength=n), out=indptr[1:])
    return indptr, nzc.astype(np.int32), x[nzr, nzc].astype(np.float32), x


def scaled(cfg: Config, n_cells: int) -> Config:
    """Same gene/cell distributions, fewer cells (bounded samples)."""
    return replace(cfg, n_cells=int(n_cells), name=f"{cfg.name}[:{n_cells}]")
