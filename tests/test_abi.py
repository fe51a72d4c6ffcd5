"""The C-ABI library builds, loads, and exports every symbol include/rsc.h declares.
No compute calls (no GPU needed); argument validation is exercised where it happens
before any CUDA call."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2603_02402_b200 import build, binding
    build.build()
    return binding.lib()


def _declared():
    text = open(os.path.join(ROOT, "include", "rsc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rsc_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    names = _declared()
    assert len(names) >= 16
    for n in names:
        assert hasattr(lib, n), f"{n} declared in rsc.h but not exported"


def test_binding_covers_header(lib):
    from paper_2603_02402_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()
    assert re.match(r"\d+\.\d+\.\d+", binding.rsc_version())


def test_struct_layout_matches_header(lib):
    from paper_2603_02402_b200 import binding as B
    assert ctypes.sizeof(B.rsc_csr) == 48
    assert B.rsc_csr.indptr.offset == 24 and B.rsc_csr.data.offset == 40
    assert ctypes.sizeof(B.rsc_outputs) == 18 * 8
    assert ctypes.sizeof(B.rsc_params) == 28
    assert ctypes.sizeof(B.rsc_filter_params) == 32 and B.rsc_filter_params.max_pct_flag.offset == 24


def test_workspace_queries(lib):
    n, G, nnz = 1000, 30000, 10**6
    assert lib.rsc_gene_moments_workspace_bytes(n, G, nnz) >= 2 * 8 * G
    assert lib.rsc_hvg_select_workspace_bytes(G, 20) >= 3 * 8 * G + 4 * G
    a = lib.rsc_preprocess_workspace_bytes(n, G, nnz, 20)
    b = lib.rsc_preprocess_host_workspace_bytes(n, G, nnz, 20)
    assert b >= a + 8 * nnz + 8 * (n + 1)
    # config 4: > 2^31 nnz must not overflow the size arithmetic
    big = lib.rsc_preprocess_host_workspace_bytes(5_000_000, 30000, 7_500_000_000, 20)
    assert big > 60 * 10**9


def test_argument_validation_before_cuda(lib):
    from paper_2603_02402_b200 import binding as B
    # NULL matrix / bad sizes are rejected on the host, with a message
    assert lib.rsc_log1p(None, None) == B.RSC_ERR_INVALID_ARG
    assert b"NULL" in lib.rsc_last_error()
    cs = B.rsc_csr(-1, 10, 0, 0, None, None, None)
    assert lib.rsc_log1p(ctypes.byref(cs), None) == B.RSC_ERR_INVALID_ARG
    cs = B.rsc_csr(4, 0, 0, 0, 1, None, None)
    assert lib.rsc_log1p(ctypes.byref(cs), None) == B.RSC_ERR_INVALID_ARG
    assert lib.rsc_hvg_select(0, None, None, 1, 20, 1, None, None, None, None, None, None, None,
                              None, 0, None) == B.RSC_ERR_INVALID_ARG
    cs = B.rsc_csr(4, 10, 0, 0, 1, None, None)
    assert lib.rsc_normalize_total(ctypes.byref(cs), -1.0, None, None, None) == B.RSC_ERR_INVALID_ARG
    assert b"target_sum" in lib.rsc_last_error()


def test_no_cpu_fallback_in_binding():
    import torch
    from paper_2603_02402_b200 import binding as B
    X = B.Csr(torch.zeros(2, dtype=torch.int64), torch.zeros(0, dtype=torch.int32),
              torch.zeros(0, dtype=torch.float32), 5)
    with pytest.raises(B.RscError):
        B.rsc_log1p(X)          # CPU tensors are refused, never silently computed


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2603_02402_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "oracle_np.py")).read()
    assert "paper_2603_02402_b200" not in osrc.split('"""', 2)[2]
