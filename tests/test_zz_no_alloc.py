"""gramsci_2pcf_noalloc (csrc/noalloc.cu): the 2pCF sweep with its accumulators in a static __device__ array instead of
allocated scratch -- for callers that cannot call cudaMalloc (CUDA graph capture, serving loops).  Compared with the
existing path (gramsci_2pcf) on calls in a row that share the array.

Collected last on purpose (the suite runs with `pytest -x`): a failure here must not hide the other tests.
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import catalogues as cat  # noqa: E402
import paper_2607_06604_b200 as gr  # noqa: E402

pytestmark = pytest.mark.gpu
RTOL_W = 1e-10      # the weighted tolerance of tests/test_gpu_parity.py (BASELINE.json: 1e-10 relative)


def _graph(seed, n, L, nb, r_max, weighted, **opts):
    import torch
    pts = cat.uniform_box(n, L, seed)
    w = np.random.default_rng(seed + 77).uniform(0.5, 1.5, n) if weighted else None
    return gr.gramsci_build_graph(torch.from_numpy(pts).cuda(), None if w is None else torch.from_numpy(w).cuda(),
                                  [L, L, L], 0.0, r_max, nb, **opts)


def _compare(g, weighted, whole=True):
    import torch
    nb = g.nbins
    c_ref, w_ref = g.pcf2(weighted=weighted)                 # the existing path (allocated scratch)
    c = torch.full((nb,), -7, dtype=torch.int64, device="cuda")
    w = torch.full((nb,), float("nan"), dtype=torch.float64, device="cuda") if weighted else None
    g.pcf2_noalloc(c, w)
    assert np.array_equal(c.cpu().numpy(), c_ref)
    assert c_ref.sum() > 0 and (not whole or c_ref.sum() == g.info()["n_edges"])
    if weighted:
        got = w.cpu().numpy()
        assert np.all(np.abs(got - w_ref) <= RTOL_W * np.abs(w_ref)), float(np.max(np.abs(got - w_ref) / np.abs(w_ref)))


def test_no_alloc_2pcf_matches_existing_path_on_calls_in_a_row():
    """Two graphs with different bin counts, alternating: every call starts from the previous call's contents in the
    shared static array and must clear them (the 17-bin result would leak into bins 6..16 of nothing -- and into bins
    0..5 of the 6-bin graph -- if it did not)."""
    import torch
    assert torch.cuda.is_available()
    ga = _graph(901, 20000, 60.0, 17, 6.0, weighted=True)
    gb = _graph(902, 6000, 40.0, 6, 5.0, weighted=True)
    gc = _graph(903, 3000, 30.0, gr.NOALLOC_MAX_BINS, 7.0, weighted=False)      # the largest size accepted
    for g, weighted in ((ga, True), (gb, True), (ga, True), (ga, False), (gc, False), (gb, True), (gb, True)):
        _compare(g, weighted)
    # a slab graph counts the edges at the hubs it owns (it also stores the halo's), as gramsci_2pcf does
    gs = _graph(901, 20000, 60.0, 17, 6.0, weighted=True, slab_count=3, slab_index=1)
    _compare(gs, True, whole=False)


def test_no_alloc_2pcf_rejects_what_would_need_an_allocation():
    import torch
    big = _graph(904, 2000, 30.0, gr.NOALLOC_MAX_BINS + 1, 6.0, weighted=False)
    out = torch.zeros(big.nbins, dtype=torch.int64, device="cuda")
    with pytest.raises(gr.GramsciError, match="GRAMSCI_NOALLOC_MAX_BINS"):
        big.pcf2_noalloc(out, None)
    g = _graph(905, 4000, 30.0, 5, 5.0, weighted=False)
    capped = _graph(905, 4000, 30.0, 5, 5.0, weighted=False, device_mem_cap_bytes=g.info()["csr_bytes"] * 2, n_windows=3)
    out = torch.zeros(5, dtype=torch.int64, device="cuda")
    with pytest.raises(gr.GramsciError, match="device-memory cap"):
        capped.pcf2_noalloc(out, None)
    host = np.zeros(5, dtype=np.int64)
    code = gr.load_library().gramsci_2pcf_noalloc(g._h, host.ctypes.data, None)
    assert code == 1 and not host.any()                                          # GRAMSCI_EINVAL, nothing written
    _compare(g, False)                                                           # and the entry point still works afterwards
