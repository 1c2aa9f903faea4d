"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Integer counts bit-exact; fp64 weighted sums within 1e-10 relative
(BASELINE.json north_star; per-bin scale = sum of |prod w|, S:8(c) A-13)."""
import os

import numpy as np
import pytest

import catalogues as cat
import oracle
import paper_2607_06604_b200 as gr

pytestmark = pytest.mark.gpu

RTOL_W = 1e-10


def _torch():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


def build_both(cfg, device_inputs=True, **opts):
    torch = _torch()
    pts, w, box = cfg["points"], cfg["weights"], cfg["box"]
    og = oracle.Graph(pts, w, box, cfg["r_min"], cfg["r_max"], cfg["nbins"])
    if device_inputs:
        dp = torch.from_numpy(pts).cuda()
        dw = None if w is None else torch.from_numpy(w).cuda()
    else:
        dp, dw = pts, w
    gg = gr.gramsci_build_graph(dp, dw, box, cfg["r_min"], cfg["r_max"], cfg["nbins"], **opts)
    return og, gg


def small(seed, n=1500, L=30.0, r_min=0.0, r_max=5.0, nb=6, weighted=False, periodic=True, snap=False):
    pts = cat.uniform_box(n, L, seed)
    if snap:
        pts = cat.snap(pts)
    w = np.random.default_rng(seed + 77).uniform(0.5, 1.5, n) if weighted else None
    return dict(points=pts, weights=w, box=[L, L, L] if periodic else None, r_min=r_min, r_max=r_max, nbins=nb)


def assert_weighted_close(got, want, scale=None):
    scale = np.abs(want) if scale is None else scale
    assert np.all(np.abs(got - want) <= RTOL_W * np.maximum(scale, 1e-300) + 0.0), \
        float(np.max(np.abs(got - want) / np.maximum(scale, 1e-300)))


@pytest.mark.parametrize("relabel", [1, 2])
@pytest.mark.parametrize("periodic,r_min,snap", [(True, 0.0, False), (False, 0.0, False), (True, 1.7, True)])
def test_graph_matches_oracle(relabel, periodic, r_min, snap):
    cfg = small(11, periodic=periodic, r_min=r_min, snap=snap)
    og, gg = build_both(cfg, relabel=relabel, want_pixels=(relabel == 2))
    o_ptr, o_idx, o_bin, o_pix = og.csr()
    if relabel == 2:
        ptr, idx, b, p = gg.export_csr(want_pix=True)
        assert np.array_equal(p, o_pix)
    else:
        ptr, idx, b = gg.export_csr()
    assert np.array_equal(ptr, o_ptr)
    assert np.array_equal(idx, o_idx)
    assert np.array_equal(b, o_bin)
    assert gg.info()["n_edges"] == og.n_edges


@pytest.mark.parametrize("relabel", [1, 2])
def test_2pcf(relabel):
    cfg = small(12, weighted=True)
    og, gg = build_both(cfg, relabel=relabel)
    oc, ow = og.pcf2()
    c, w = gg.pcf2(weighted=True)
    assert np.array_equal(c, oc)
    assert_weighted_close(w, ow)


ALGOS = [gr.ALGO_DEFAULT, gr.ALGO_MERGEPATH, gr.ALGO_BSEARCH, gr.ALGO_BITMAP, gr.ALGO_TABLE_G1, gr.ALGO_TABLE_G2,
         gr.ALGO_TABLE_G4, gr.ALGO_TABLE_G8, gr.ALGO_GATHER]


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("relabel", [1, 2])
def test_3pcf_config1(relabel, algo):
    cfg = cat.config1()
    if relabel == 2 and algo == gr.ALGO_GATHER:        # the dense rows need labels in cell order
        _, gg = build_both(cfg, relabel=relabel, algo=algo)
        with pytest.raises(gr.GramsciError) as e:
            gg.pcf3()
        assert e.value.code == 2
        return
    og, gg = build_both(cfg, relabel=relabel, algo=algo)
    oc, _ = og.pcf3()
    c, _ = gg.pcf3()
    assert c.sum() == oc.sum()
    assert np.array_equal(c, oc)
    # host-buffer path gives the same
    c2, _ = gg.pcf3(host=True)
    assert np.array_equal(c2, oc)


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("periodic,r_min", [(True, 0.0), (False, 0.0), (True, 2.0)])
def test_3pcf_weighted(periodic, r_min, algo):
    cfg = small(13, n=4000, L=40.0, weighted=True, periodic=periodic, r_min=r_min, nb=7)
    og, gg = build_both(cfg, device_inputs=False, algo=algo)
    oc, ow = og.pcf3()
    c, w = gg.pcf3(weighted=True)
    assert np.array_equal(c, oc)
    assert_weighted_close(w, ow)


@pytest.mark.parametrize("algo", ALGOS)
def test_histogram_drain_path_exact(algo, monkeypatch):
    """The shared-memory uint32 histograms are drained into the global uint64 ones when a hit budget is passed
    (2^28 per warp / 0xF0000000 per CTA by default: only the largest workload gets there).  With the budget forced
    down to a few thousand hits every kernel variant drains hundreds of times on small inputs; every bin must
    still equal the oracle's."""
    monkeypatch.setenv("GRAMSCI_FLUSH_BUDGET", "3000")
    cfg = cat.config1()
    og, gg = build_both(cfg, algo=algo)
    assert np.array_equal(gg.pcf3()[0], og.pcf3()[0])
    cfg = cat.config2_data(seed=2102, n=8_000, L=200.0, mean_parents=80.0)
    og, gg = build_both(cfg, algo=algo)
    oc, ow = og.pcf3()
    c, w = gg.pcf3(weighted=True)
    assert c.sum() > 1e6 and np.array_equal(c, oc)
    assert_weighted_close(w, ow)
    cfg, oc = _bao_replica()
    gg = gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], algo=algo)
    assert np.array_equal(gg.pcf3()[0], oc)


@pytest.mark.parametrize("budget", ["", "2500"])
def test_weighted_fixed_point_limbs(budget, monkeypatch):
    """GRAMSCI_WMODE=1: weighted sums of the gather kernels as 13-bit fixed-point limbs in shared memory (order-
    independent) instead of fp64 RED atomics -- same 1e-10 bar, short and long rows, capped graph."""
    monkeypatch.setenv("GRAMSCI_WMODE", "1")
    if budget:
        monkeypatch.setenv("GRAMSCI_FLUSH_BUDGET", budget)
    for cfg in (small(13, n=4000, L=40.0, weighted=True, nb=7), cat.config2_data(seed=2103, n=12_000, L=230.0, mean_parents=120.0)):
        og, gg = build_both(cfg, algo=gr.ALGO_GATHER)
        oc, ow = og.pcf3()
        c, w = gg.pcf3(weighted=True)
        assert np.array_equal(c, oc)
        assert_weighted_close(w, ow)
        w2 = gg.pcf3(counts=False, weighted=True)[1]       # weights only (no count plane in shared memory)
        assert_weighted_close(w2, ow)
    cfg = cat.config5(seed=5102, n=3_000, L=310.0)          # rows of ~1,500 entries: CTA kernel, drains inside a hub
    w = np.random.default_rng(9).uniform(0.5, 1.5, 3000)
    og = oracle.Graph(cfg["points"], w, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    gg = gr.gramsci_build_graph(cfg["points"], w, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], algo=gr.ALGO_GATHER)
    c, ws = gg.pcf3(weighted=True)
    assert gg.info()["max_row"] > 800 and np.array_equal(c, og.pcf3()[0])
    assert_weighted_close(ws, og.pcf3()[1])


def test_4pcf_lut_drain_path_exact(monkeypatch):
    monkeypatch.setenv("GRAMSCI_FLUSH_BUDGET", "2000")
    monkeypatch.setenv("GRAMSCI_4PCF_LUT", "1")
    cfg = cat.config4(seed=4002, n=6000, cap_deg=7.0)
    og, gg = build_both(cfg, want_pixels=True)
    ec, ew, oc, ow = og.pcf4(parity=True)
    gec, goc, gew, gow = gg.pcf4_parity(weighted=True)
    assert ec.sum() > 10000 and np.array_equal(gec, ec) and np.array_equal(goc, oc)
    assert_weighted_close(gew, ew)
    assert_weighted_close(gow, ow, scale=np.abs(ew))


def test_torch_allocator_hooks():
    """S:8(b): gramsci_options.alloc / dealloc -- the graph and all scratch from PyTorch's caching allocator."""
    torch = _torch()
    cfg = small(71, n=5000, L=40.0, weighted=True, r_max=5.0, nb=5)
    og = oracle.Graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    torch.cuda.synchronize()
    torch.cuda.reset_peak_memory_stats()
    before = torch.cuda.memory_allocated()
    g = gr.gramsci_build_graph(torch.from_numpy(cfg["points"]).cuda(), torch.from_numpy(cfg["weights"]).cuda(), cfg["box"],
                               cfg["r_min"], cfg["r_max"], cfg["nbins"], torch_allocator=True)
    held = torch.cuda.memory_allocated() - before
    assert held >= 5 * og.n_edges            # the CSR lives in torch's allocator
    c, w = g.pcf3(weighted=True)
    assert np.array_equal(c, og.pcf3()[0])
    assert_weighted_close(w, og.pcf3()[1])
    assert np.array_equal(g.pcf4()[0], og.pcf4()[0])
    g.free()
    assert torch.cuda.memory_allocated() - before < held
    gr.gramsci_release_memory()


def test_concurrent_builds_on_two_threads():
    """include/gramsci.h THREADS: no process-global device state -- two host threads build and query different
    graphs (different boxes, radii and bin counts) on their own streams at the same time."""
    import threading
    torch = _torch()
    cfgs = [small(81, n=20000, L=60.0, r_max=5.0, nb=6), small(82, n=15000, L=33.0, r_min=1.0, r_max=4.0, nb=9, periodic=False)]
    want = [oracle.Graph(c["points"], None, c["box"], c["r_min"], c["r_max"], c["nbins"]) for c in cfgs]
    want = [(o.n_edges, o.pcf2()[0], o.pcf3()[0]) for o in want]
    got = [None, None]
    errs = []

    def work(k):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                c = cfgs[k]
                pts = torch.from_numpy(c["points"]).cuda()
                res = []
                for _ in range(6):
                    g = gr.gramsci_build_graph(pts, None, c["box"], c["r_min"], c["r_max"], c["nbins"])
                    res.append((g.info()["n_edges"], g.pcf2()[0], g.pcf3()[0]))
                    g.free()
                got[k] = res
        except Exception as e:           # noqa: BLE001
            errs.append(e)

    th = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    [t.start() for t in th]
    [t.join() for t in th]
    assert not errs, errs
    for k in range(2):
        for e, c2, c3 in got[k]:
            assert e == want[k][0] and np.array_equal(c2, want[k][1]) and np.array_equal(c3, want[k][2])


def test_range_errors_on_very_long_rows():
    """GRAMSCI_ERANGE paths: a row too long for the kernel's shared-memory staging (66,000 mutually adjacent points:
    rows of up to 65,999 entries, 2.2e9 edges).  Raised before any enumeration starts."""
    torch = _torch()
    if torch.cuda.mem_get_info()[0] < 40 * 2 ** 30:
        pytest.skip("needs 40 GiB of free device memory")
    n = 66_000
    pts = np.random.default_rng(5).random((n, 3)) * 0.5 + 10.0
    g = gr.gramsci_build_graph(torch.from_numpy(pts).cuda(), None, None, 0.0, 1.0, 3)
    assert g.info()["max_row"] == n - 1 and g.info()["n_edges"] == n * (n - 1) // 2
    assert g.pcf2()[0].sum() == n * (n - 1) // 2
    with pytest.raises(gr.GramsciError) as e:
        g.pcf4()
    assert e.value.code == 2
    for algo in (gr.ALGO_BSEARCH, gr.ALGO_MERGEPATH, gr.ALGO_BITMAP):
        ga = gr.gramsci_build_graph(torch.from_numpy(pts).cuda(), None, None, 0.0, 1.0, 3, algo=algo)
        with pytest.raises(gr.GramsciError) as e:
            ga.pcf3()
        assert e.value.code == 2
        ga.free()


def _diag(h, nb):
    return np.array([h.reshape(nb, nb, nb)[b, b, b] for b in range(nb)])


@pytest.mark.parametrize("opts", [dict(), dict(algo=gr.ALGO_GATHER), dict(algo=gr.ALGO_BSEARCH), dict(relabel=2),
                                  dict(relabel=2, hub_stride=3)])
def test_3pcf_equilateral(opts):
    """S:8(f)-3 (the equilateral 3pCF is one of the four query kernels): triangles with all three edges
    in one radial bin, restricted inside the kernel, against the diagonal of the oracle's full 3pCF -- the gather
    kernels (short rows, long rows), the search-kernel fallback (caller labels), weighted, and under a memory cap."""
    stride = opts.get("hub_stride", 1)
    cfg = cat.config1()
    og, gg = build_both(cfg, **opts)
    oc, _ = og.pcf3(hubs=(0, og.n, stride))
    c, _ = gg.pcf3_equilateral()
    assert c.shape == (cfg["nbins"],) and c.sum() > 1000
    assert np.array_equal(c, _diag(oc, cfg["nbins"]))
    assert np.array_equal(gg.pcf3_equilateral(host=True)[0], c)
    # clustered replica of configs[1], weighted
    cfg = cat.config2_data(seed=2104, n=15_625, L=250.0, mean_parents=156.25)
    og, gg = build_both(cfg, **opts)
    oc, ow = og.pcf3(hubs=(0, og.n, stride))
    c, w = gg.pcf3_equilateral(weighted=True)
    assert c.sum() > 1e5 and np.array_equal(c, _diag(oc, cfg["nbins"]))
    assert_weighted_close(w, _diag(ow, cfg["nbins"]))
    if stride == 1:
        # the same graph under a device-memory cap (windows streamed from host memory)
        csr = gg.info()["csr_bytes"]
        _, gc = build_both(cfg, device_mem_cap_bytes=int(csr * 4), n_windows=4, **opts)
        c2, w2 = gc.pcf3_equilateral(weighted=True)
        assert gc.info()["n_windows"] == 4 and np.array_equal(c2, c)
        assert_weighted_close(w2, _diag(ow, cfg["nbins"]))
        # rows of thousands of entries, r_min > 0
        cfg, oc = _bao_replica()
        gb = gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], **opts)
        assert np.array_equal(gb.pcf3_equilateral()[0], _diag(oc, cfg["nbins"]))


def test_edge_cases():
    torch = _torch()
    # empty catalogue, single point, no edges, one triangle
    for pts in (np.zeros((0, 3)), np.array([[0.5, 0.5, 0.5]]), np.array([[0.1, 0.1, 0.1], [5.0, 5.0, 5.0]])):
        g = gr.gramsci_build_graph(pts, None, [10.0, 10.0, 10.0], 0.0, 1.0, 3)
        assert g.info()["n_edges"] == 0
        c, _ = g.pcf3(host=True)
        assert c.sum() == 0
        c2, _ = g.pcf2(host=True)
        assert c2.sum() == 0
        assert g.pcf3_equilateral(host=True)[0].sum() == 0
    tri = np.array([[1.0, 1.0, 1.0], [1.5, 1.0, 1.0], [1.0, 1.9, 1.0]])
    g = gr.gramsci_build_graph(tri, None, None, 0.0, 3.0, 3)
    og = oracle.Graph(tri, None, None, 0.0, 3.0, 3)
    c, _ = g.pcf3(host=True)
    assert np.array_equal(c, og.pcf3()[0]) and c.sum() == 1
    # coincident points are an edge iff r_min == 0 (A-6)
    dup = np.array([[1.0, 1.0, 1.0], [1.0, 1.0, 1.0], [1.2, 1.0, 1.0]])
    for r_min in (0.0, 0.1):
        g = gr.gramsci_build_graph(dup, None, None, r_min, 1.0, 2)
        og = oracle.Graph(dup, None, None, r_min, 1.0, 2)
        assert g.info()["n_edges"] == og.n_edges
        assert np.array_equal(g.pcf3(host=True)[0], og.pcf3()[0])
    # periodic box with fewer than three cells per axis (stencil aliasing)
    cfg = small(14, n=600, L=10.0, r_max=4.5, nb=4)
    og, gg = build_both(cfg)
    assert np.array_equal(gg.pcf3()[0], og.pcf3()[0])
    # errors
    with pytest.raises(gr.GramsciError) as e:
        gr.gramsci_build_graph(cfg["points"], None, [10.0, 10.0, 10.0], 0.0, 5.0, 4)
    assert e.value.code == 2


# ---- 4pCF and parity-decomposed 4pCF (S:8(a) A8-A10) --------------------------------------------------
@pytest.mark.parametrize("relabel", [1, 2])
@pytest.mark.parametrize("periodic,r_min,nb", [(True, 0.0, 4), (False, 0.0, 6), (True, 1.5, 3)])
def test_4pcf(relabel, periodic, r_min, nb):
    cfg = small(21, n=3000, L=30.0, weighted=True, periodic=periodic, r_min=r_min, r_max=5.0, nb=nb)
    og, gg = build_both(cfg, relabel=relabel)
    oc, ow = og.pcf4()
    assert oc.sum() > 1000
    c, w = gg.pcf4(weighted=True)
    assert np.array_equal(c, oc)
    assert_weighted_close(w, ow)
    # counts only, straight into host memory
    c2, _ = gg.pcf4(host=True)
    assert np.array_equal(c2, oc)
    # the disconnected term needs the 2pCF of the same graph (Eq. 4, A-12)
    assert np.array_equal(gg.pcf2()[0], og.pcf2()[0])


@pytest.mark.parametrize("periodic", [True, False])
def test_4pcf_parity(periodic):
    cfg = small(22, n=3000, L=30.0, weighted=True, periodic=periodic, r_max=5.0, nb=5)
    og, gg = build_both(cfg, want_pixels=True)
    ec, ew, oc, ow = og.pcf4(parity=True)
    assert np.abs(oc).sum() > 100
    gec, goc, gew, gow = gg.pcf4_parity(weighted=True)
    assert np.array_equal(gec, ec)
    assert np.array_equal(goc, oc)
    assert_weighted_close(gew, ew)
    assert_weighted_close(gow, ow, scale=np.abs(ew))      # A-13: scale = sum |prod w| of the bin
    # even channel == plain 4pCF; parity needs pixels and caller labels
    assert np.array_equal(gg.pcf4()[0], ec)
    _, g2 = build_both(cfg)
    with pytest.raises(gr.GramsciError) as e:
        g2.pcf4_parity()
    assert e.value.code == 1
    with pytest.raises(gr.GramsciError) as e:       # pixels are oriented by caller label (A-10)
        build_both(cfg, want_pixels=True, relabel=1)
    assert e.value.code == 1


@pytest.mark.parametrize("lut", ["0", "1"])
def test_4pcf_parity_wedge(lut, monkeypatch):
    """Scaled replica of BASELINE configs[3] (survey wedge, open box, weights U(0.8,1.2), 8 bins); with the
    plain raw-histogram kernel and with the opt-in configuration-LUT variant (GRAMSCI_4PCF_LUT=1)."""
    monkeypatch.setenv("GRAMSCI_4PCF_LUT", lut)
    cfg = cat.config4(seed=4002, n=6000, cap_deg=7.0)
    og, gg = build_both(cfg, want_pixels=True)
    ec, ew, oc, ow = og.pcf4(parity=True)
    assert ec.sum() > 10000
    gec, goc, gew, gow = gg.pcf4_parity(weighted=True)
    assert np.array_equal(gec, ec)
    assert np.array_equal(goc, oc)
    assert_weighted_close(gew, ew)
    assert_weighted_close(gow, ow, scale=np.abs(ew))


def test_4pcf_injection_on_gpu():
    """P:261 injection idea on the CUDA path: isolated scalene tetrahedra, mirrored fraction 30 %."""
    r_min, r_max, nb = 4.0, 10.0, 6
    tet = cat.tetra_from_lengths(*cat.SCALENE_EDGES)
    K = 200
    mirror = np.zeros(K, dtype=bool)
    mirror[: int(0.3 * K)] = True
    pts, _, _ = cat.isolated_units(tet, K, spacing=40.0, seed=91, mirror_mask=mirror)
    og = oracle.Graph(pts, None, None, r_min, r_max, nb)
    gg = gr.gramsci_build_graph(pts, None, None, r_min, r_max, nb, want_pixels=True)
    ec, _, oc, _ = og.pcf4(parity=True)
    gec, goc, _, _ = gg.pcf4_parity()
    i6 = np.ravel_multi_index((0, 1, 2, 3, 4, 5), (nb,) * 6)
    assert gec[i6] == K and gec.sum() == K
    assert np.array_equal(gec, ec) and np.array_equal(goc, oc)
    assert abs(goc[i6] - (K - 2 * int(mirror.sum()))) <= 0.04 * K


def test_4pcf_edge_cases():
    _torch()
    for pts in (np.zeros((0, 3)), np.array([[0.5, 0.5, 0.5]]), np.array([[1.0, 1.0, 1.0], [1.5, 1.0, 1.0], [1.0, 1.9, 1.0]])):
        g = gr.gramsci_build_graph(pts, None, None, 0.0, 3.0, 2, want_pixels=True)
        ec, oc, _, _ = g.pcf4_parity(host=True)
        assert ec.sum() == 0 and not oc.any()
    # one regular tetrahedron -> one 4-clique in bin (0,0,0,0,0,0)
    tet = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=np.float64) * 0.3 + 5.0
    g = gr.gramsci_build_graph(tet, None, None, 0.0, 3.0, 3)
    c, _ = g.pcf4(host=True)
    assert c.sum() == 1 and c[0] == 1
    with pytest.raises(gr.GramsciError):
        gr.gramsci_build_graph(tet, None, None, 0.0, 3.0, 17).pcf4()


# ---- larger / clustered shapes and the out-of-core tiler (S:8(a) A11; pin C-13) -----------------------------
@pytest.mark.parametrize("algo", [gr.ALGO_DEFAULT, gr.ALGO_MERGEPATH, gr.ALGO_BSEARCH, gr.ALGO_TABLE_G4])
def test_3pcf_clustered_replica(algo):
    """1/64 replica of BASELINE configs[1] data (Neyman-Scott, same densities, fp64 weights)."""
    cfg = cat.config2_data(seed=2101, n=15_625, L=250.0, mean_parents=156.25)
    og, gg = build_both(cfg, algo=algo)
    oc, ow = og.pcf3()
    c, w = gg.pcf3(weighted=True)
    assert c.sum() > 5e6
    assert np.array_equal(c, oc)
    assert_weighted_close(w, ow)


_BAO = {}


def _bao_replica():
    if not _BAO:
        cfg = cat.config5(seed=5101, n=6_000, L=310.0)
        og = oracle.Graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
        _BAO["cfg"], _BAO["cnt"] = cfg, og.pcf3()[0]
    return _BAO["cfg"], _BAO["cnt"]


@pytest.mark.parametrize("algo", [gr.ALGO_DEFAULT, gr.ALGO_MERGEPATH, gr.ALGO_BSEARCH, gr.ALGO_TABLE_G8])
def test_3pcf_bao_replica(algo):
    """Shrunk replica of BASELINE configs[4] (same radii and bins, L=310, 40 % of the density so that
    the oracle finishes in seconds): rows of thousands of entries, r_min > 0, 18 bins, a periodic grid
    with two cells per axis."""
    cfg, oc = _bao_replica()
    gg = gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], algo=algo)
    c, _ = gg.pcf3()
    assert gg.info()["max_row"] > 2000 and oc.sum() > 1e9
    assert np.array_equal(c, oc)


@pytest.mark.parametrize("kmajor", ["1", "0"])
def test_gather_cta_loop_orders(kmajor, monkeypatch):
    """The long-row gather kernel in both loop orders (GRAMSCI_CTA_KMAJOR=1: lanes keep their tail entries and loop
    over the spokes, the default; 0: one spoke per warp, tail streamed): counts, fp64 weighted sums and the
    equilateral restriction against the oracle, with small spoke tiles and histogram drains forced."""
    monkeypatch.setenv("GRAMSCI_CTA_KMAJOR", kmajor)
    cfg, oc = _bao_replica()
    for tile_mb, budget in (("", ""), ("1", "2500")):
        if tile_mb:
            monkeypatch.setenv("GRAMSCI_TILE_MB", tile_mb)
            monkeypatch.setenv("GRAMSCI_FLUSH_BUDGET", budget)
        gg = gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], algo=gr.ALGO_GATHER)
        assert gg.info()["max_row"] > 2000
        assert np.array_equal(gg.pcf3()[0], oc)
        assert np.array_equal(gg.pcf3_equilateral()[0], oc.reshape(18, 18, 18)[np.arange(18), np.arange(18), np.arange(18)])
    # slab + halo graphs on long rows (hub range inside the CTA kernel): two slabs add up
    tot = np.zeros_like(oc)
    for rank in range(2):
        gs = gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], algo=gr.ALGO_GATHER,
                                    slab_count=2, slab_index=rank)
        tot += gs.pcf3()[0]
    assert np.array_equal(tot, oc)
    c5 = cat.config5(seed=5102, n=3_000, L=310.0)
    w = np.random.default_rng(9).uniform(0.5, 1.5, 3000)
    og = oracle.Graph(c5["points"], w, c5["box"], c5["r_min"], c5["r_max"], c5["nbins"])
    gw = gr.gramsci_build_graph(c5["points"], w, c5["box"], c5["r_min"], c5["r_max"], c5["nbins"], algo=gr.ALGO_GATHER)
    c, ws = gw.pcf3(weighted=True)
    o_c, o_w = og.pcf3()
    assert gw.info()["max_row"] > 800 and np.array_equal(c, o_c)
    assert_weighted_close(ws, o_w)


@pytest.mark.parametrize("relabel", [1, 2])
@pytest.mark.parametrize("n_windows,cap_frac", [(2, 1.2), (5, 1.0), (7, 0.45)])
def test_out_of_core_equals_in_core(relabel, n_windows, cap_frac):
    """C-13: the capped (windowed, streamed from pinned host memory) run is bit-identical to the in-core
    run for any window count, including windows forced small on a tiny input."""
    cfg = small(31, n=6000, L=40.0, weighted=True, r_max=5.0, nb=5)
    og, g0 = build_both(cfg, relabel=relabel)
    oc, ow = og.pcf3()
    csr = g0.info()["csr_bytes"]
    _, g1 = build_both(cfg, relabel=relabel, device_mem_cap_bytes=int(csr * cap_frac), n_windows=n_windows)
    assert g1.info()["n_windows"] == n_windows and g1.info()["n_edges"] == og.n_edges
    c, w = g1.pcf3(weighted=True)
    assert np.array_equal(c, oc)
    assert np.array_equal(c, g0.pcf3()[0])
    assert_weighted_close(w, ow)
    assert g1.timing(4) >= csr * 0.99            # every window was staged at least once
    c2, w2 = g1.pcf2(weighted=True)
    assert np.array_equal(c2, og.pcf2()[0])


@pytest.mark.parametrize("n_windows", [2, 5, 9])
def test_out_of_core_gather_kernel(n_windows, monkeypatch):
    """The gather kernel under a device-memory cap: a window buffer holds the CSR rows and the dense cell-block rows
    expanded from them on the device; hubs of window h against spokes of window c.  Forced
    (GRAMSCI_ALGO_GATHER), so a fall-back to another kernel would be an error; also with the long-row (CTA) kernel and
    its spoke tiles, and through the histogram drains."""
    cfg = small(33, n=6000, L=40.0, weighted=True, r_max=5.0, nb=5)
    og, g0 = build_both(cfg)
    oc, ow = og.pcf3()
    csr = g0.info()["csr_bytes"]
    _, g1 = build_both(cfg, device_mem_cap_bytes=int(csr * 4.0), n_windows=n_windows, algo=gr.ALGO_GATHER)
    assert g1.info()["n_windows"] == n_windows
    c, w = g1.pcf3(weighted=True)
    assert np.array_equal(c, oc)
    assert_weighted_close(w, ow)
    assert g1.timing(4) >= csr * 0.99
    monkeypatch.setenv("GRAMSCI_FLUSH_BUDGET", "2500")
    monkeypatch.setenv("GRAMSCI_TILE_MB", "1")
    cfg2, oc2 = _bao_replica()
    gb = gr.gramsci_build_graph(cfg2["points"], None, cfg2["box"], cfg2["r_min"], cfg2["r_max"], cfg2["nbins"],
                                algo=gr.ALGO_GATHER, n_windows=n_windows, device_mem_cap_bytes=2 ** 31)
    assert gb.info()["n_windows"] == n_windows
    assert np.array_equal(gb.pcf3()[0], oc2)


def test_out_of_core_cap_derives_windows():
    cfg = small(32, n=8000, L=40.0, r_max=5.0, nb=4)
    og, g0 = build_both(cfg)
    csr = g0.info()["csr_bytes"]
    _, g1 = build_both(cfg, device_mem_cap_bytes=csr // 2)
    assert g1.info()["n_windows"] >= 8           # four window buffers must fit under the cap
    assert np.array_equal(g1.pcf3()[0], og.pcf3()[0])
    assert np.array_equal(g1.pcf4()[0], og.pcf4()[0])      # 4pCF tiles over (h, c1 <= c2)


@pytest.mark.parametrize("relabel,n_windows", [(1, 2), (1, 3), (1, 6), (2, 4)])
def test_out_of_core_4pcf_equals_in_core(relabel, n_windows):
    """under a memory cap the 4pCF runs over tiles (hub window h, search windows c1 <= c2); every tetrahedron
    lands in exactly one tile, so counts equal the resident run and the oracle bit for bit (C-13), weighted sums to
    A-13's tolerance.  relabel=2 keeps caller labels (every window reaches every window)."""
    cfg = small(35, n=5000, L=36.0, weighted=True, r_max=5.0, nb=4)
    og, g0 = build_both(cfg, relabel=relabel)
    oc, ow = og.pcf4()
    csr = g0.info()["csr_bytes"]
    _, g1 = build_both(cfg, relabel=relabel, device_mem_cap_bytes=int(csr * 2.0), n_windows=n_windows)
    assert g1.info()["n_windows"] == n_windows
    c, w = g1.pcf4(weighted=True)
    assert c.sum() == oc.sum() > 0
    assert np.array_equal(c, oc)
    assert np.array_equal(c, g0.pcf4()[0])
    assert_weighted_close(w, ow)
    assert g1.timing(4) >= csr * 0.99


@pytest.mark.parametrize("n_windows", [3, 5])
def test_out_of_core_4pcf_parity_equals_in_core(n_windows):
    """The parity-decomposed 4pCF (caller labels, pixel bytes staged with the hub window) under a cap: all four
    channels against the oracle."""
    c4 = cat.config4(seed=4005, n=4000, cap_deg=6.0)
    o4 = oracle.Graph(c4["points"], c4["weights"], None, c4["r_min"], c4["r_max"], c4["nbins"])
    rec, rew, roc, row = o4.pcf4(parity=True)
    g0 = gr.gramsci_build_graph(c4["points"], c4["weights"], None, c4["r_min"], c4["r_max"], c4["nbins"], want_pixels=True)
    csr = g0.info()["csr_bytes"]
    g1 = gr.gramsci_build_graph(c4["points"], c4["weights"], None, c4["r_min"], c4["r_max"], c4["nbins"], want_pixels=True,
                                device_mem_cap_bytes=int(csr * 2.0), n_windows=n_windows)
    assert g1.info()["n_windows"] == n_windows
    ec, oc, ew, ow = g1.pcf4_parity(weighted=True)
    assert ec.sum() == rec.sum() > 0
    assert np.array_equal(ec, rec) and np.array_equal(oc, roc)
    assert np.all(np.abs(ew - rew) <= 1e-10 * np.abs(rew)) and np.all(np.abs(ow - row) <= 1e-10 * np.abs(rew))


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times ------------------------------------
@pytest.mark.slow
@pytest.mark.parametrize("which", ["cfg2R", "cfg2D"])
def test_full_size_config2_matches_oracle(which):
    """configs[1] in full (1e6 points per catalogue, device-resident inputs, default algo = what bench.py
    times): every bin of the 3pCF against the full oracle run (about 10 s of host time on 16 cores)."""
    cfg = cat.config2_randoms() if which == "cfg2R" else cat.config2_data()
    og, gg = build_both(cfg)
    assert gg.info()["n_edges"] == og.n_edges
    oc, ow = og.pcf3()
    weighted = cfg["weights"] is not None
    c, w = gg.pcf3(weighted=weighted)
    assert c.sum() == oc.sum() and np.array_equal(c, oc)
    if weighted:
        assert_weighted_close(w, ow)
    assert np.array_equal(gg.pcf2()[0], og.pcf2()[0])


@pytest.mark.slow
def test_full_size_config3_matches_oracle():
    """configs[2] in full (2e5 points, 1.5e9 tetrahedra): every bin of the 4pCF, the 3pCF and the 2pCF of the
    same graph against the full oracle run; relabelling invariance (C-3) on the GPU path at full size; the
    total on the Monte-Carlo 4-clique density of a Poisson field (C-6)."""
    cfg = cat.config3()
    og = oracle.Graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    oc, _ = og.pcf4()
    gg = gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    c, _ = gg.pcf4()
    assert c.sum() == oc.sum() > 1e9
    assert np.array_equal(c, oc)
    assert np.array_equal(gg.pcf3()[0], og.pcf3()[0])
    assert np.array_equal(gg.pcf2()[0], og.pcf2()[0])
    perm = np.random.default_rng(7).permutation(og.n)
    g2 = gr.gramsci_build_graph(np.ascontiguousarray(cfg["points"][perm]), None, cfg["box"], cfg["r_min"],
                                cfg["r_max"], cfg["nbins"])
    assert np.array_equal(g2.pcf4()[0], c)
    # Poisson 4-clique density: N m^3 p4 / 24 with p4 = 0.1582 +- 0.0002 (Monte Carlo)
    m = 2.0 * og.n_edges / og.n
    assert abs(c.sum() / (og.n * m ** 3 * 0.1582 / 24.0) - 1.0) < 0.01


@pytest.mark.slow
def test_full_size_config4_replica_parity_matches_oracle():
    """Reduced configs[3] (62,500 points in a 15 x 15 degree wedge -- an eighth of the points in a quarter of the
    solid angle, i.e. half the density -- same radii, bins and weights U(0.8,1.2); 2.1e10 tetrahedra): all four
    channels of the parity-decomposed 4pCF against the full oracle."""
    cfg = cat.config4(n=62_500, cap_deg=15.0)
    og = oracle.Graph(cfg["points"], cfg["weights"], None, cfg["r_min"], cfg["r_max"], cfg["nbins"])
    ec, ew, oc, ow = og.pcf4(parity=True)
    gg = gr.gramsci_build_graph(cfg["points"], cfg["weights"], None, cfg["r_min"], cfg["r_max"], cfg["nbins"],
                                want_pixels=True)
    gec, goc, gew, gow = gg.pcf4_parity(weighted=True)
    assert gec.sum() == ec.sum() > 1e10
    assert np.array_equal(gec, ec) and np.array_equal(goc, oc)
    assert_weighted_close(gew, ew)
    assert_weighted_close(gow, ow, scale=np.abs(ew))


@pytest.mark.slow
def test_full_size_config4_parity_sampled_hubs():
    """configs[3] in full (5e5 points, 1.54e12 tetrahedra, weighted, even and odd channels).  The full oracle run
    would take more than an hour of host time, so the oracle enumerates the tetrahedra whose smallest-label vertex
    is a multiple of 128 and the CUDA path is asked for exactly that partial result (``hub_stride``), on the graph
    and in the launch configuration of the full run; the full run itself must contain the partial one."""
    cfg = cat.config4()
    stride = 128
    og = oracle.Graph(cfg["points"], cfg["weights"], None, cfg["r_min"], cfg["r_max"], cfg["nbins"])
    ec, ew, oc, ow = og.pcf4(parity=True, hubs=(0, og.n, stride))
    pts = _torch().from_numpy(cfg["points"]).cuda()
    w = _torch().from_numpy(cfg["weights"]).cuda()
    gs = gr.gramsci_build_graph(pts, w, None, cfg["r_min"], cfg["r_max"], cfg["nbins"], want_pixels=True, hub_stride=stride)
    assert gs.info()["n_edges"] == og.n_edges
    gec, goc, gew, gow = gs.pcf4_parity(weighted=True)
    assert gec.sum() == ec.sum() > 5e9
    assert np.array_equal(gec, ec) and np.array_equal(goc, oc)
    assert_weighted_close(gew, ew)
    assert_weighted_close(gow, ow, scale=np.abs(ew))
    # the same graph without the hub filter = what bench.py --workload cfg4 times
    gf = gr.gramsci_build_graph(pts, w, None, cfg["r_min"], cfg["r_max"], cfg["nbins"], want_pixels=True)
    fec, foc, few, fow = gf.pcf4_parity(weighted=True)
    assert fec.sum() > 1e12 and np.all(fec >= gec) and np.all(few >= gew * (1 - 1e-12))
    big = fec > 50_000_000
    assert big.sum() > 100 and np.allclose(gec[big] / fec[big], 1.0 / stride, rtol=0.1)
    # 3pCF and 2pCF of the same (caller-label) graph against the oracle, hub-sampled and in full
    assert np.array_equal(gs.pcf3()[0], og.pcf3(hubs=(0, og.n, stride))[0])
    assert np.array_equal(gf.pcf2()[0], og.pcf2()[0])


def test_hub_stride_partial_results():
    cfg = small(41, n=3000, L=30.0, weighted=True, r_max=5.0, nb=4)
    og = oracle.Graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    for algo in (gr.ALGO_DEFAULT, gr.ALGO_MERGEPATH, gr.ALGO_BSEARCH, gr.ALGO_TABLE_G4):
        g = gr.gramsci_build_graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"],
                                   relabel=2, hub_stride=7, algo=algo)
        assert np.array_equal(g.pcf3()[0], og.pcf3(hubs=(0, og.n, 7))[0])
        assert np.array_equal(g.pcf4()[0], og.pcf4(hubs=(0, og.n, 7))[0])
        assert np.array_equal(g.export_labels(), np.arange(og.n))
    # spatial (cell-order) labels: the stride applies to the INTERNAL label; the oracle sees the points in internal
    # order (gramsci_export_labels), where its labels are the library's
    for algo in (gr.ALGO_DEFAULT, gr.ALGO_GATHER, gr.ALGO_BITMAP, gr.ALGO_BSEARCH, gr.ALGO_MERGEPATH):
        g = gr.gramsci_build_graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"],
                                   hub_stride=5, algo=algo)
        lab = g.export_labels()
        assert np.array_equal(np.sort(lab), np.arange(og.n))
        oi = oracle.Graph(cfg["points"][lab], cfg["weights"][lab], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
        c, w = g.pcf3(weighted=True)
        oc, ow = oi.pcf3(hubs=(0, og.n, 5))
        assert 0 < oc.sum() < og.pcf3()[0].sum()
        assert np.array_equal(c, oc)
        assert_weighted_close(w, ow)
        # the on-demand walk written for graphs too large to hold (what the full configs[4] test uses)
        od = oracle.Graph(cfg["points"][lab], cfg["weights"][lab], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"],
                          lists=False)
        assert np.array_equal(od.pcf3_direct(np.arange(0, og.n, 5))[0], oc)


def test_ddd_over_rrr_poisson_is_one():
    """BASELINE north_star: for Poisson points in a periodic box DDD/RRR -> 1 within shot noise.  Two independent
    uniform catalogues through the CUDA path and the host estimator helper (NNN/RRR per configuration)."""
    from paper_2607_06604_b200 import estimators as est
    n, L, nb = 60_000, 300.0, 6
    d = cat.uniform_box(n, L, 61)
    r = cat.uniform_box(2 * n, L, 62)
    gd = gr.gramsci_build_graph(d, None, [L, L, L], 0.0, 20.0, nb)
    grr = gr.gramsci_build_graph(r, None, [L, L, L], 0.0, 20.0, nb)
    cd, _ = gd.pcf3()
    cr, _ = grr.pcf3()
    zeta = est.zeta3_ratio(cd, n, cr, 2 * n)
    ok = cd > 20_000
    assert ok.sum() >= 20
    # relative scatter of a triangle count ~ a few / sqrt(count) (triples share pairs)
    assert np.all(np.abs(zeta[ok] - 1.0) < 12.0 / np.sqrt(cd[ok]) + 12.0 / np.sqrt(cr[ok]))
    assert abs(np.nansum(cd) / n ** 3 / (np.nansum(cr) / (2 * n) ** 3) - 1.0) < 5e-3


@pytest.mark.slow
def test_full_size_config5_invariants_and_cap():
    """configs[4] in full (2.5e6 points, 8.4e9 edges, 42 GB of CSR, 7.1e12 triangles; about two minutes on a
    B200).  No oracle run is feasible at this size, so the result is checked through properties that hold at
    any size: pair and triangle counts per configuration on their Poisson expectations (C-6; a periodic
    uniform box), and the run under a 24 GiB device-memory cap bit-identical to the resident run (C-13)."""
    torch = _torch()
    free, _ = torch.cuda.mem_get_info()
    try:
        host_gb = os.sysconf("SC_PHYS_PAGES") * os.sysconf("SC_PAGE_SIZE") / 2 ** 30
    except (ValueError, OSError):
        host_gb = 0.0
    if free < 70 * 2 ** 30 or host_gb < 80:
        pytest.skip("needs 70 GiB of free device memory and 80 GiB of host memory")
    cfg = cat.config5()
    n, L, nb = cfg["points"].shape[0], float(cfg["box"][0]), cfg["nbins"]
    pts = torch.from_numpy(cfg["points"]).cuda()
    g = gr.gramsci_build_graph(pts, None, cfg["box"], cfg["r_min"], cfg["r_max"], nb)
    e = cfg["r_min"] + np.arange(nb + 1) * (cfg["r_max"] - cfg["r_min"]) / nb
    V = L ** 3
    c2, _ = g.pcf2()
    exp2 = 0.5 * n * (n - 1) * (4 * np.pi / 3) * (e[1:] ** 3 - e[:-1] ** 3) / V
    assert c2.sum() == g.info()["n_edges"] > 8.3e9
    assert np.all(np.abs(c2 / exp2 - 1.0) < 5e-4)
    c3, _ = g.pcf3()
    g.free()
    c3r = c3.reshape(nb, nb, nb)
    I = (e[1:] ** 2 - e[:-1] ** 2) / 2
    worst, checked = 0.0, 0
    for a in range(nb):
        for b in range(a, nb):
            for c in range(b, nb):
                assert c3r[b, a, c] == 0 or a == b                     # populated at sorted triples only (A-5)
                if e[c + 1] <= e[a] + e[b]:                             # triangle inequality holds on the whole bins
                    mu = 6 if a < b < c else (1 if a == c else 3)
                    exp3 = n * (n - 1) * (n - 2) / 6 / V ** 2 * mu * 8 * np.pi ** 2 * I[a] * I[b] * I[c]
                    worst = max(worst, abs(c3r[a, b, c] / exp3 - 1.0))
                    checked += 1
    assert checked > 1000 and worst < 2e-3, (checked, worst)
    assert 7.0e12 < c3.sum() < 7.2e12
    g2 = gr.gramsci_build_graph(pts, None, cfg["box"], cfg["r_min"], cfg["r_max"], nb, device_mem_cap_bytes=24 * 2 ** 30)
    assert g2.info()["n_windows"] >= 4
    c3c, _ = g2.pcf3()
    assert g2.timing(4) > 40e9                                          # the windows really were streamed
    assert np.array_equal(c3c, c3)
    g2.free()
    # EXACT check in the launch configuration bench.py times (spatial labels, default kernel; 2^28-hit histogram
    # drains are reached here): the triangles whose smallest-INTERNAL-label vertex is a multiple of `stride`, against
    # the oracle's on-demand walk over the same points given in internal order (gramsci_export_labels)
    stride = 8192
    gs = gr.gramsci_build_graph(pts, None, cfg["box"], cfg["r_min"], cfg["r_max"], nb, hub_stride=stride)
    lab = gs.export_labels()
    cs, _ = gs.pcf3()
    gs.free()
    od = oracle.Graph(cfg["points"][lab], None, cfg["box"], cfg["r_min"], cfg["r_max"], nb, lists=False)
    oc, _ = od.pcf3_direct(np.arange(0, n, stride))
    assert oc.sum() > 5e8
    assert np.array_equal(cs, oc)
    assert np.all(c3 >= cs)


def test_hub_shards_add_up_to_the_full_result():
    """S:8(e): the hubs of one catalogue sharded over `shard_count` devices; the shard histograms sum to the full
    result (exactly for counts) -- here the shards run one after the other on one GPU."""
    cfg = small(51, n=4000, L=32.0, weighted=True, r_max=5.0, nb=5)
    og = oracle.Graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    oc3, ow3 = og.pcf3()
    ec, ew, oc, ow = og.pcf4(parity=True)
    for world in (2, 3):
        c3 = np.zeros_like(oc3); w3 = np.zeros_like(ow3)
        gec = np.zeros_like(ec); goc = np.zeros_like(oc); gew = np.zeros_like(ew); gow = np.zeros_like(ow)
        for rank in range(world):
            g = gr.gramsci_build_graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"],
                                       shard_count=world, shard_index=rank)
            c, w = g.pcf3(weighted=True)
            assert 0 < c.sum() < oc3.sum()
            c3 += c; w3 += w
            gp = gr.gramsci_build_graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"],
                                        want_pixels=True, shard_count=world, shard_index=rank)
            a, b, cc, d = gp.pcf4_parity(weighted=True)
            gec += a; goc += b; gew += cc; gow += d
        assert np.array_equal(c3, oc3) and np.array_equal(gec, ec) and np.array_equal(goc, oc)
        assert_weighted_close(w3, ow3)
        assert_weighted_close(gew, ew)
        assert_weighted_close(gow, ow, scale=np.abs(ew))
    with pytest.raises(gr.GramsciError):
        gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], shard_count=2, shard_index=2)


@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("algo", [0, 2, 3])
def test_slab_and_halo_partition_adds_up(periodic, algo):
    """S:8(e): one slab of cells per device, each holding only the rows of its slab and of the halo its
    hubs' spokes live in.  The slabs own disjoint hub ranges covering the catalogue, every slab stores fewer edges
    than the full graph, and the 2pCF / 3pCF / 4pCF histograms of the slabs sum to the oracle's (counts exactly) --
    here the slabs run one after the other on one GPU; also under a memory cap (windows) per slab."""
    cfg = small(53, n=12000, L=60.0, weighted=True, r_max=5.0, nb=5, periodic=periodic)
    og = oracle.Graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    oc2, ow2 = og.pcf2()
    oc3, ow3 = og.pcf3()
    oc4, ow4 = og.pcf4()
    n = cfg["points"].shape[0]
    for world in (2, 5):
        c2 = np.zeros_like(oc2); w2 = np.zeros_like(ow2); c3 = np.zeros_like(oc3); w3 = np.zeros_like(ow3)
        c4 = np.zeros_like(oc4); w4 = np.zeros_like(ow4); cc3 = np.zeros_like(oc3); cc4 = np.zeros_like(oc4)
        cover, stored = [], []
        for rank in range(world):
            g = gr.gramsci_build_graph(cfg["points"], cfg["weights"], cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"],
                                       slab_count=world, slab_index=rank, algo=algo)
            cover.append(g.slab_range())
            stored.append(g.info()["n_edges"])
            a, b = g.pcf2(weighted=True); c2 += a; w2 += b
            a, b = g.pcf3(weighted=True); c3 += a; w3 += b
            a, b = g.pcf4(weighted=True); c4 += a; w4 += b
            csr = g.info()["csr_bytes"]
            g.free()
            gc = gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"],
                                        slab_count=world, slab_index=rank, algo=algo, device_mem_cap_bytes=max(csr, 4096) * 2,
                                        n_windows=3)
            cc3 += gc.pcf3()[0]
            if world == 2:                                           # 4pCF tiles (h, c1 <= c2) on a capped slab graph
                cc4 += gc.pcf4()[0]
            gc.free()
        assert cover[0][0] == 0 and cover[-1][1] == n and all(cover[k][1] == cover[k + 1][0] for k in range(world - 1))
        assert all(hi > lo for lo, hi in cover)                      # every slab got hubs (work-balanced cut)
        assert max(stored) < og.n_edges and sum(stored) >= og.n_edges
        if world == 5:
            assert max(stored) < 0.6 * og.n_edges                    # slab + halo, not the whole graph
        assert np.array_equal(c2, oc2) and np.array_equal(c3, oc3) and np.array_equal(c4, oc4) and np.array_equal(cc3, oc3)
        assert world != 2 or np.array_equal(cc4, oc4)
        assert_weighted_close(w2, ow2); assert_weighted_close(w3, ow3); assert_weighted_close(w4, ow4)
    with pytest.raises(gr.GramsciError):                             # needs cell-order labels
        gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], slab_count=2, relabel=2)
    with pytest.raises(gr.GramsciError):
        gr.gramsci_build_graph(cfg["points"], None, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], slab_count=2, shard_count=2)


def test_many_bins_global_histogram_path():
    """nb^3 bins beyond shared memory (40^3 x 4 B = 256 KB): the search kernel with a global histogram."""
    cfg = small(61, n=2500, L=30.0, weighted=True, r_max=6.0, nb=40)
    og, gg = build_both(cfg)
    oc, ow = og.pcf3()
    c, w = gg.pcf3(weighted=True)
    assert np.array_equal(c, oc)
    assert_weighted_close(w, ow)
    cfg1 = small(62, n=1500, L=30.0, r_min=2.0, r_max=6.0, nb=1)
    og1, gg1 = build_both(cfg1)
    assert np.array_equal(gg1.pcf3()[0], og1.pcf3()[0]) and np.array_equal(gg1.pcf4()[0], og1.pcf4()[0])


def test_signed_weights():
    """A-13: data-minus-random style weights of both signs; judged against sum |prod w| per bin."""
    cfg = small(63, n=3000, L=30.0, r_max=5.0, nb=5)
    rng = np.random.default_rng(64)
    w = rng.uniform(0.5, 1.5, 3000) * rng.choice([-1.0, 1.0], 3000)
    og = oracle.Graph(cfg["points"], w, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    oa = oracle.Graph(cfg["points"], np.abs(w), cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"])
    for opts in (dict(), dict(algo=gr.ALGO_BSEARCH), dict(algo=gr.ALGO_MERGEPATH)):
        gg = gr.gramsci_build_graph(cfg["points"], w, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], **opts)
        c, ws = gg.pcf3(weighted=True)
        assert np.array_equal(c, og.pcf3()[0])
        assert_weighted_close(ws, og.pcf3()[1], scale=oa.pcf3()[1])
        c2, w2 = gg.pcf2(weighted=True)
        assert_weighted_close(w2, og.pcf2()[1], scale=oa.pcf2()[1])
    gp = gr.gramsci_build_graph(cfg["points"], w, cfg["box"], cfg["r_min"], cfg["r_max"], cfg["nbins"], want_pixels=True)
    ec, oc, ew, ow = gp.pcf4_parity(weighted=True)
    rec, rew, roc, row = og.pcf4(parity=True)
    sc = oa.pcf4()[1]
    assert np.array_equal(ec, rec) and np.array_equal(oc, roc)
    assert_weighted_close(ew, rew, scale=sc)
    assert_weighted_close(ow, row, scale=sc)


# ---- estimator layer end to end (S:8(f)-1) ---------------------------------------------------------
def test_signed_combined_catalogue_is_dd_minus_2dr_plus_rr():
    """with data weights summing to +1 and random weights to -1, the weighted pair sum of the COMBINED catalogue
    in a bin is DD/N_D^2 - 2 DR/(N_D N_R) + RR/N_R^2.  DD, RR (separate graphs) and DR (combined minus both) are
    integer counts from the unweighted path, so this pins the signed fp64 path -- where the terms cancel to a few
    per cent of their size -- by exact integers.  The 3pCF of the combined catalogue against the oracle, judged on
    the A-13 scale sum |prod w|."""
    from paper_2607_06604_b200 import estimators as est
    d = cat.config2_data(seed=2105, n=20_000, L=270.0, mean_parents=200.0)
    r = cat.config2_randoms(seed=2106, n=30_000, L=270.0)
    nd, nr = d["points"].shape[0], r["points"].shape[0]
    pts, w, wr = est.combined_catalogue(d["points"], r["points"])
    assert abs(w[:nd].sum() - 1.0) < 1e-12 and abs(w[nd:].sum() + 1.0) < 1e-12
    box, rmin, rmax, nb = d["box"], d["r_min"], d["r_max"], d["nbins"]
    gd = gr.gramsci_build_graph(d["points"], None, box, rmin, rmax, nb)
    grr = gr.gramsci_build_graph(r["points"], None, box, rmin, rmax, nb)
    gc = gr.gramsci_build_graph(pts, w, box, rmin, rmax, nb)
    dd, rr = gd.pcf2()[0], grr.pcf2()[0]
    cc, nn = gc.pcf2(weighted=True)
    dr = cc - dd - rr
    want = dd / nd ** 2 - dr / (nd * nr) + rr / nr ** 2
    scale = dd / nd ** 2 + dr / (nd * nr) + rr / nr ** 2              # sum |w_i w_j|
    assert np.all(np.abs(want[-5:]) < 0.1 * scale[-5:])                  # at large r the terms cancel to a few per cent
    assert np.all(np.abs(nn - want) <= 1e-10 * scale)
    xi = est.signed_ratio(nn, rr / nr ** 2)
    assert np.all(xi[:4] > 1.0)                                          # a clustered catalogue: xi >> 0 at small r
    # triplets: combined signed catalogue against the oracle (sum |prod w| from the |w| run)
    og = oracle.Graph(pts, w, box, rmin, rmax, nb)
    oa = oracle.Graph(pts, np.abs(w), box, rmin, rmax, nb)
    c3, n3 = gc.pcf3(weighted=True)
    assert np.array_equal(c3, og.pcf3()[0])
    assert_weighted_close(n3, og.pcf3()[1], scale=oa.pcf3()[1])


@pytest.mark.slow
def test_estimators_on_poisson_catalogues_at_full_size():
    """configs[1] / configs[2] shapes through the estimator layer on the GPU path, Poisson data so that the truth is
    known: (i) the combined 2e6-point signed catalogue (uniform "data" + uniform randoms in the configs[1] box): NNN/RRR
    = 0 within shot noise -- the cancellation stress of the fp64 weighted path at full size; (ii) configs[2] points as
    data + an equal-size random catalogue: NNNN/RRRR (even channel), xi = NN/RR, zeta_disc from Eq. 4 and zeta_conn =
    zeta - zeta_disc (Eq. 5) all consistent with 0."""
    from paper_2607_06604_b200 import estimators as est
    torch = _torch()
    # (i) 3pCF, 1e6 + 1e6 points, r < 30, 15 bins
    d = cat.config2_randoms(seed=2201)
    r = cat.config2_randoms(seed=2202)
    nr = r["points"].shape[0]
    pts, w, _ = est.combined_catalogue(d["points"], r["points"])
    box, rmin, rmax, nb = d["box"], d["r_min"], d["r_max"], d["nbins"]
    gc = gr.gramsci_build_graph(torch.from_numpy(pts).cuda(), torch.from_numpy(w).cuda(), box, rmin, rmax, nb)
    grr = gr.gramsci_build_graph(torch.from_numpy(r["points"]).cuda(), None, box, rmin, rmax, nb)
    c3, nnn = gc.pcf3(weighted=True)
    rrr = grr.pcf3()[0] / float(nr) ** 3
    gc.free(); grr.free()
    ok = rrr * float(nr) ** 3 > 1e5
    zeta = est.signed_ratio(nnn, rrr)
    # a signed triple sum is a sum of ~8x as many +-terms as RRR has triangles; its noise is ~ a few / sqrt(RRR)
    assert ok.sum() > 300 and np.all(np.abs(zeta[ok]) < 60.0 / np.sqrt(rrr[ok] * float(nr) ** 3))
    assert c3.sum() > 7.5e9                                              # ~8x the triangles of one catalogue
    # (ii) 4pCF, configs[2] + randoms
    d = cat.config3()
    r = cat.config3(seed=3002)
    nr = r["points"].shape[0]
    pts, w, _ = est.combined_catalogue(d["points"], r["points"])
    box, rmin, rmax, nb = d["box"], d["r_min"], d["r_max"], d["nbins"]
    gc = gr.gramsci_build_graph(torch.from_numpy(pts).cuda(), torch.from_numpy(w).cuda(), box, rmin, rmax, nb)
    grr = gr.gramsci_build_graph(torch.from_numpy(r["points"]).cuda(), None, box, rmin, rmax, nb)
    c4, nnnn = gc.pcf4(weighted=True)
    rc4 = grr.pcf4()[0]
    nn = gc.pcf2(weighted=True)[1]
    rc2 = grr.pcf2()[0]
    rr = rc2 / float(nr) ** 2
    rrrr = rc4 / float(nr) ** 4
    xi = est.signed_ratio(nn, rr)
    assert np.all(np.abs(xi) < 8.0 / np.sqrt(rc2))                      # DD - 2DR + RR: shot noise ~ 2 / sqrt(RR)
    zeta = est.signed_ratio(nnnn, rrrr)
    zconn = est.zeta4_connected(np.nan_to_num(zeta), xi)
    ok = rc4 > 2e5
    assert ok.sum() > 500 and c4.sum() > 2e10
    assert np.all(np.abs(zeta[ok]) < 100.0 / np.sqrt(rc4[ok]))
    assert np.all(np.abs(zconn[ok]) < 100.0 / np.sqrt(rc4[ok]) + 1e-4)


@pytest.mark.parametrize("seed", [11, 12])
def test_randomized_shapes_and_options(seed, monkeypatch):
    """A seeded sweep over graph shapes (density, radii, bin counts, periodic / open, clustered / uniform, signed weights) and
    library options (kernel variant, capped windows, slab and modulo shards, caller labels, forced drains and spoke tiles):
    2pCF, 3pCF, equilateral 3pCF and 4pCF against the oracle -- counts bit for bit, weighted sums to A-13's tolerance.
    (GRAMSCI_FUZZ_CASES=n runs n cases per seed instead of 25; 2 x 4,000 cases pass on the final build, and an earlier
    run of this sweep found the two-window 4pCF tiling bug fixed in csrc/tiler.cu.)"""
    torch = _torch()
    rng = np.random.default_rng(seed)
    done, cases = 0, int(os.environ.get("GRAMSCI_FUZZ_CASES", "25"))
    while done < cases:
        periodic = bool(rng.integers(2))
        nb = int(rng.choice([1, 2, 3, 5, 6, 9, 15, 18]))
        L = float(rng.choice([20.0, 33.0, 47.0]))
        r_max = float(rng.uniform(2.0, min(8.0, 0.49 * L)))
        r_min = float(rng.choice([0.0, 0.0, rng.uniform(0.0, 0.6 * r_max)]))
        n = int(min(max(50, float(rng.choice([0.02, 0.08, 0.3, 0.6])) * L ** 3), 12000))
        if rng.integers(3) == 0:
            pts = cat.config2_data(seed=int(rng.integers(1 << 30)), n=n, L=L, mean_parents=max(3.0, n / 80.0))["points"]
        else:
            pts = cat.uniform_box(n, L, int(rng.integers(1 << 30)))
        weighted = bool(rng.integers(2))
        w = rng.uniform(0.5, 1.5, n) if weighted else None
        if weighted and rng.integers(4) == 0:
            w = w * rng.choice([-1.0, 1.0], n)
        box = [L, L, L] if periodic else None
        og = oracle.Graph(pts, w, box, r_min, r_max, nb)
        if og.n_edges == 0 or og.n_edges > 1.2e6:
            continue
        algo = int(rng.choice([0, 0, 0, 1, 2, 3]))
        mode = int(rng.integers(6))
        for key, val in (("GRAMSCI_FLUSH_BUDGET", str(int(rng.choice([700, 3000, 20000]))) if rng.integers(3) == 0 else None),
                         ("GRAMSCI_TILE_MB", "1" if rng.integers(4) == 0 else None),
                         ("GRAMSCI_CTA_KMAJOR", str(int(rng.integers(2))) if rng.integers(3) == 0 else None),
                         ("GRAMSCI_WMODE", "1" if rng.integers(5) == 0 else None)):
            if val is None:
                monkeypatch.delenv(key, raising=False)
            else:
                monkeypatch.setenv(key, val)
        if mode == 1:
            graphs = [dict(device_mem_cap_bytes=8 * 5 * og.n_edges + 65536, n_windows=int(rng.integers(2, 8)))]
        elif mode == 2 and algo != 1:
            k = int(rng.integers(2, 6))
            graphs = [dict(slab_count=k, slab_index=r) for r in range(k)]
        elif mode == 3:
            k = int(rng.integers(2, 5))
            graphs = [dict(shard_count=k, shard_index=r) for r in range(k)]
        elif mode == 4:
            graphs = [dict(relabel=2)]
        elif mode == 5:
            graphs = [dict(want_pixels=True)]
        else:
            graphs = [dict()]
        what = dict(periodic=periodic, nb=nb, L=L, r_min=r_min, r_max=r_max, n=n, weighted=weighted, algo=algo, graphs=graphs)
        oc2, _ = og.pcf2()
        oc3, ow3 = og.pcf3()
        do4 = nb <= 6 and og.n_edges < 1.5e5
        if do4:
            oc4, ow4 = og.pcf4()
        c2 = np.zeros_like(oc2); c3 = np.zeros_like(oc3); w3 = np.zeros_like(ow3); ce = np.zeros(nb, dtype=np.int64)
        c4 = np.zeros(nb ** 6, dtype=np.int64); w4 = np.zeros(nb ** 6)
        for gopt in graphs:
            g = gr.gramsci_build_graph(torch.from_numpy(pts).cuda(), None if w is None else torch.from_numpy(w).cuda(), box,
                                       r_min, r_max, nb, algo=algo, **gopt)
            c2 += g.pcf2()[0]
            a, b = g.pcf3(weighted=weighted)
            c3 += a
            if weighted:
                w3 += b
            ce += g.pcf3_equilateral()[0]
            if do4:
                a, b = g.pcf4(weighted=weighted)
                c4 += a
                if weighted:
                    w4 += b
            if do4 and mode == 5:                                    # parity split: all four channels (A-8 ... A-11)
                ec, oc, ew, ow = g.pcf4_parity(weighted=weighted)
                rec, rew, roc, row = og.pcf4(parity=True)
                assert np.array_equal(ec, rec) and np.array_equal(oc, roc), what
                if weighted:
                    sc4 = oracle.Graph(pts, np.abs(w), box, r_min, r_max, nb).pcf4()[1]
                    assert_weighted_close(ew, rew, scale=sc4)
                    assert_weighted_close(ow, row, scale=sc4)
            g.free()
        assert mode == 3 or np.array_equal(c2, oc2), what            # (2pCF is not sharded by shard_count)
        assert np.array_equal(c3, oc3), what
        assert np.array_equal(ce, oc3.reshape(nb, nb, nb)[np.arange(nb), np.arange(nb), np.arange(nb)]), what
        if do4:
            assert np.array_equal(c4, oc4), what
        if weighted:
            oabs = oracle.Graph(pts, np.abs(w), box, r_min, r_max, nb)       # A-13: judged against sum |prod w|
            assert_weighted_close(w3, ow3, scale=oabs.pcf3()[1])
            if do4:
                assert_weighted_close(w4, ow4, scale=oabs.pcf4()[1])
        done += 1
