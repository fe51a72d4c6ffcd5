"""rsc_hvg_select_no_alloc: rsc_hvg_select on the library's built-in device scratch
array, for callers that cannot allocate.  Checked against the existing entry point (which is checked
against the oracle in test_gpu_parity.py) on two calls in a row with different inputs -- the calls
share the scratch array, so the second one must not see anything of the first -- and against the
oracle itself.  Collected last on purpose (file name): the suite runs with pytest -x.
"""
import numpy as np
import pytest
import torch

from oracle import oracle_np as O
import parity_util as U

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2603_02402_b200 import build, binding
    build.build()
    binding.lib()


def _moments(G, seed):
    """Seeded per-gene mean / variance with the degenerate genes HVG has to cope with."""
    rng = np.random.default_rng(seed)
    mean = np.exp(rng.normal(-1.5, 1.5, G))
    var = mean * np.exp(rng.normal(0.3, 0.6, G))
    mean[::97] = 0.0
    var[::97] = 0.0                                        # all-zero genes: NaN dispersion
    var[5::211] = 0.0                                      # constant genes
    return mean, var


KEYS_EXACT = ("bin", "mask", "count")
KEYS_F64 = ("mean_t", "disp", "disp_norm")


def _compare(a, b, tag):
    for k in KEYS_EXACT:
        assert torch.equal(a[k], b[k]), f"{tag}: {k} differs from rsc_hvg_select"
    n = int(a["count"].item())
    assert torch.equal(a["indices"][:n], b["indices"][:n]), f"{tag}: indices differ"
    for k in KEYS_F64:                                     # same kernels, same inputs: bit-identical
        assert np.array_equal(U.np_(a[k]), U.np_(b[k]), equal_nan=True), f"{tag}: {k} differs"


@pytest.mark.parametrize("hvg_single_cta", [0, 1])
def test_two_calls_in_a_row_match_the_workspace_path(hvg_single_cta):
    from paper_2603_02402_b200 import binding as B
    B.rsc_set_option("hvg_single_cta", hvg_single_cta)
    try:
        calls = [(30000, 4000, 20, 11), (1800, 200, 7, 12), (65536, 5000, 20, 13)]
        for i, (G, n_top, n_bins, seed) in enumerate(calls):
            mean, var = _moments(G, seed)
            m, v = torch.as_tensor(mean).cuda(), torch.as_tensor(var).cuda()
            want = B.rsc_hvg_select(m, v, n_top, n_bins)
            got = B.rsc_hvg_select_no_alloc(m, v, n_top, n_bins)
            torch.cuda.synchronize()
            _compare(got, want, f"call {i} (G={G})")
            ref = O.hvg_select(mean, var, n_top, n_bins)
            U.assert_hvg_matches(got, ref, n_top, f"call {i} vs oracle", strict=False)
        # only the required outputs: the optional arrays then live in the scratch array
        G, n_top, n_bins, seed = calls[0]
        mean, var = _moments(G, seed)
        m, v = torch.as_tensor(mean).cuda(), torch.as_tensor(var).cuda()
        want = B.rsc_hvg_select(m, v, n_top, n_bins)
        out = dict(mask=torch.empty(G, dtype=torch.uint8, device="cuda"),
                   count=torch.zeros(1, dtype=torch.int32, device="cuda"))
        got = B.rsc_hvg_select_no_alloc(m, v, n_top, n_bins, out=out)
        torch.cuda.synchronize()
        assert torch.equal(got["mask"], want["mask"]) and torch.equal(got["count"], want["count"])
    finally:
        B.rsc_set_option("hvg_single_cta", 0)


def test_limit_is_enforced_and_nothing_is_allocated():
    from paper_2603_02402_b200 import binding as B
    lim = B.rsc_hvg_select_no_alloc_max_genes()
    assert lim == 65536
    G = lim + 1
    m = torch.ones(G, dtype=torch.float64, device="cuda")
    with pytest.raises(B.RscError) as e:
        B.rsc_hvg_select_no_alloc(m, m, 10)
    assert "exceeds the built-in scratch" in str(e.value)
    # the call itself takes no device memory: free memory as the driver reports it does not move
    # across calls once the outputs exist (the first call above already looked the array up)
    G = 20000
    mean, var = _moments(G, 3)
    m, v = torch.as_tensor(mean).cuda(), torch.as_tensor(var).cuda()
    out = B.rsc_hvg_select_no_alloc(m, v, 2000)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        B.rsc_hvg_select_no_alloc(m, v, 2000, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
