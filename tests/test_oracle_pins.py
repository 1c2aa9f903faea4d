"""Pins for the CPU oracle (SURVEY.md 8(c) C-1 ... C-12): everything here runs without a GPU and
checks ``oracle/`` against things other than itself -- brute force written twice (C and NumPy, with
different formulas), SciPy / NumPy library routines, Poisson closed forms, isolated rigid units with
analytically known counts, invariances, and the configuration counts the paper prints."""
import itertools
import math
import os

import numpy as np
import pytest
import scipy.sparse as sp
from scipy.spatial import cKDTree

import catalogues
import oracle
from oracle import brute_numpy as bn

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def small_cfg(seed, n=220, L=10.0, r_min=0.0, r_max=3.0, nb=5, weighted=True, periodic=True):
    rng = np.random.default_rng(seed)
    pts = rng.random((n, 3)) * L
    w = rng.uniform(0.5, 1.5, size=n) if weighted else None
    return pts, w, ([L, L, L] if periodic else None), r_min, r_max, nb


# ------------------------------------------------------------------------------------------
# graph: edge set vs a library routine (cKDTree with periodic boxsize) and vs all-pairs

@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("r_min", [0.0, 1.2])
def test_graph_edges_match_kdtree(periodic, r_min):
    pts, w, box, _, r_max, nb = small_cfg(11, n=1500, L=20.0, r_max=2.5, periodic=periodic)
    g = oracle.Graph(pts, None, box, r_min, r_max, nb)
    start, idx, b, _ = g.csr()
    tree = cKDTree(pts, boxsize=(box[0] if periodic else None))
    big = tree.query_pairs(r_max, output_type="ndarray")
    small = tree.query_pairs(r_min, output_type="ndarray") if r_min > 0 else np.zeros((0, 2), dtype=np.int64)
    want = {tuple(sorted(p)) for p in big.tolist()} - {tuple(sorted(p)) for p in small.tolist()}
    rows = np.repeat(np.arange(g.n), np.diff(start))
    got = set(zip(rows.tolist(), idx.tolist()))
    assert got == want
    # rows sorted ascending, oriented (Eq. 1, A-15)
    for i in range(g.n):
        r = idx[start[i]:start[i + 1]]
        assert np.all(np.diff(r) > 0) and (r.size == 0 or r[0] > i)
    # cells vs all-pairs construction: identical CSR
    g2 = oracle.Graph(pts, None, box, r_min, r_max, nb, use_cells=False)
    for a, c in zip(g.csr(), g2.csr()):
        assert np.array_equal(a, c)


@pytest.mark.parametrize("periodic", [True, False])
def test_degrees_direct_match_kdtree(periodic):
    """og_degrees_direct (rows found on demand from the cell list, graph built with lists=False): full degree
    against cKDTree ball counts (a library routine), oriented degree against the row lengths of the stored CSR."""
    pts, w, box, _, r_max, nb = small_cfg(13, n=1200, L=20.0, r_max=2.5, periodic=periodic)
    r_min = 0.8
    g = oracle.Graph(pts, None, box, r_min, r_max, nb)
    gd = oracle.Graph(pts, None, box, r_min, r_max, nb, lists=False)
    labels = np.arange(0, g.n, 7)
    full, plus = gd.degrees_direct(labels)
    start, idx, _, _ = g.csr()
    assert np.array_equal(plus, np.diff(start)[labels])
    tree = cKDTree(pts, boxsize=(box[0] if periodic else None))
    big = tree.query_pairs(r_max, output_type="ndarray")
    small = tree.query_pairs(r_min, output_type="ndarray")
    deg = np.bincount(big.ravel(), minlength=g.n) - np.bincount(small.ravel(), minlength=g.n)
    assert np.array_equal(full, deg[labels])


def test_bin_byte_matches_sqrt_floor():
    pts, w, box, r_min, r_max, nb = small_cfg(12, n=800, L=15.0, r_min=0.5, r_max=3.0, nb=7)
    g = oracle.Graph(pts, None, box, r_min, r_max, nb)
    start, idx, b, pix = g.csr()
    bm, d = bn.adjacency(pts, box, r_min, r_max, nb)
    rows = np.repeat(np.arange(g.n), np.diff(start))
    assert np.array_equal(bm[rows, idx], b.astype(np.int64))
    assert np.array_equal(bn.pixel_of(d[rows, idx]), pix.astype(np.int64))


def test_invalid_arguments():
    pts = np.random.default_rng(0).random((10, 3))
    with pytest.raises(ValueError):
        oracle.Graph(pts, None, [1.0, 1.0, 1.0], 0.0, 0.5, 4)      # r_max >= L/2 (A-4)
    with pytest.raises(ValueError):
        oracle.Graph(pts, None, None, 0.3, 0.2, 4)
    with pytest.raises(ValueError):
        oracle.Graph(pts, None, None, 0.0, 0.2, 0)


# ------------------------------------------------------------------------------------------
# C-1: brute force (C and NumPy) == neighbour-list walks, bit for bit on counts

@pytest.mark.parametrize("seed,periodic,r_min", [(1, True, 0.0), (2, False, 0.0), (3, True, 0.9)])
def test_c1_brute_vs_walks(seed, periodic, r_min):
    pts, w, box, _, r_max, nb = small_cfg(seed, n=160, L=9.0, r_max=3.0, nb=4, periodic=periodic)
    g = oracle.Graph(pts, w, box, r_min, r_max, nb)
    # 2pCF
    c2, w2 = g.pcf2()
    c2b, w2b = g.pcf2(brute=True)
    c2n, w2n = bn.pcf2(pts, w, box, r_min, r_max, nb)
    assert np.array_equal(c2, c2b) and np.array_equal(c2, c2n)
    assert np.allclose(w2, w2b, rtol=1e-13) and np.allclose(w2, w2n, rtol=1e-13)
    # 3pCF
    c3, w3 = g.pcf3()
    c3b, w3b = g.pcf3(brute=True)
    c3n, w3n = bn.pcf3(pts, w, box, r_min, r_max, nb)
    assert c3.sum() > 100
    assert np.array_equal(c3, c3b) and np.array_equal(c3, c3n)
    assert np.allclose(w3, w3b, rtol=1e-13) and np.allclose(w3, w3n, rtol=1e-13)
    # 4pCF + parity
    ec, ew, oc, ow = g.pcf4(parity=True)
    ecb, ewb, ocb, owb = g.pcf4(parity=True, brute=True)
    ecn, ewn, ocn, own = bn.pcf4(pts, w, box, r_min, r_max, nb, parity=True)
    assert ec.sum() > 50
    assert np.array_equal(ec, ecb) and np.array_equal(ec, ecn)
    assert np.array_equal(oc, ocb) and np.array_equal(oc, ocn)
    assert np.allclose(ew, ewb, rtol=1e-13) and np.allclose(ew, ewn, rtol=1e-13)
    assert np.allclose(ow, owb, rtol=1e-12, atol=1e-12) and np.allclose(ow, own, rtol=1e-12, atol=1e-12)
    # plain 4pCF == even channel
    e2c, e2w = g.pcf4(parity=False)
    assert np.array_equal(e2c, ec) and np.allclose(e2w, ew, rtol=1e-13)
    # only canonical positions are populated
    n3, cfg3 = oracle.num_configs(3, nb, want_list=True)
    mask3 = np.zeros(nb ** 3, bool)
    mask3[(cfg3[:, 0] * nb + cfg3[:, 1]) * nb + cfg3[:, 2]] = True
    assert not c3[~mask3].any()
    n4, cfg4 = oracle.num_configs(4, nb, want_list=True)
    mask4 = np.zeros(nb ** 6, bool)
    mask4[np.ravel_multi_index(cfg4.T, (nb,) * 6)] = True
    assert not ec[~mask4].any() and not oc[~mask4].any()


# ------------------------------------------------------------------------------------------
# C-2: totals == clique counts of the graph from library routines

def test_c2_totals_are_clique_counts():
    pts, w, box, r_min, r_max, nb = small_cfg(21, n=900, L=12.0, r_max=2.8, nb=6)
    g = oracle.Graph(pts, None, box, r_min, r_max, nb)
    start, idx, _, _ = g.csr()
    rows = np.repeat(np.arange(g.n), np.diff(start))
    U = sp.csr_matrix((np.ones(idx.size, dtype=np.int64), (rows, idx)), shape=(g.n, g.n))
    n_tri = int((U @ U).multiply(U).sum())
    A = (U + U.T).toarray().astype(np.float64)
    assert n_tri == round(np.trace(A @ A @ A) / 6.0)            # trace(A^3)/6
    c3, _ = g.pcf3()
    assert int(c3.sum()) == n_tri
    # 4-cliques: sum over edges of (#edges inside the common neighbourhood) / 6
    k4 = 0
    for i, j in zip(rows.tolist(), idx.tolist()):
        c = A[i] * A[j]
        k4 += float(c @ A @ c) / 2.0
    k4 = round(k4 / 6.0)
    e4, _ = g.pcf4()
    assert int(e4.sum()) == k4 and k4 > 1000
    c2, _ = g.pcf2()
    assert int(c2.sum()) == idx.size


# ------------------------------------------------------------------------------------------
# C-3 / C-4: relabelling, rigid motions, mirror

def _all_stats(pts, w, box, r_min, r_max, nb):
    g = oracle.Graph(pts, w, box, r_min, r_max, nb)
    return g.pcf2() + g.pcf3() + g.pcf4(parity=True)


def test_c3_relabelling_invariance():
    pts, w, box, r_min, r_max, nb = small_cfg(31, n=400, L=10.0, r_max=2.6, nb=4)
    ref = _all_stats(pts, w, box, r_min, r_max, nb)
    p = np.random.default_rng(5).permutation(len(pts))
    got = _all_stats(pts[p], w[p], box, r_min, r_max, nb)
    for k, (a, b) in enumerate(zip(ref, got)):
        if k in (6, 7):
            continue        # odd channel: label-dependent through the pixelised hub choice (A-10)
        if a.dtype == np.int64:
            assert np.array_equal(a, b)
        else:
            assert np.allclose(a, b, rtol=1e-12)


def test_c4_translation_axis_permutation_and_mirror():
    rng = np.random.default_rng(41)
    L = 16.0
    pts = catalogues.snap(rng.random((500, 3)) * L)              # 2^-10 grid: d2 exact in fp64
    args = (None, [L, L, L], 0.0, 3.0, 5)
    ref = _all_stats(pts, *args)
    shift = np.array([3.25, 7.0, 11.5])                          # grid multiples
    moved = np.mod(pts + shift, L)
    got = _all_stats(moved, *args)
    for k in (0, 2, 4):                                          # counts: 2pCF, 3pCF, even 4pCF
        assert np.array_equal(ref[k], got[k])
    got = _all_stats(pts[:, [2, 0, 1]], *args)
    for k in (0, 2, 4):
        assert np.array_equal(ref[k], got[k])
    # mirror x -> -x in an open box: every count identical, odd -> -odd exactly (A-8 grid symmetric)
    pts = rng.random((500, 3)) * 8.0
    w = rng.uniform(0.5, 1.5, size=500)
    ref = _all_stats(pts, w, None, 0.0, 2.5, 4)
    mir = pts.copy()
    mir[:, 0] *= -1.0
    got = _all_stats(mir, w, None, 0.0, 2.5, 4)
    for k in (0, 2, 4):
        assert np.array_equal(ref[k], got[k])
    assert np.array_equal(ref[6], -got[6]) and np.any(ref[6] != 0)
    assert np.allclose(ref[7], -got[7], rtol=1e-12, atol=1e-12)


# ------------------------------------------------------------------------------------------
# C-5: rebinning -- nb bins summed pairwise == nb/2 bins ("rebinned exactly")

def test_c5_rebinning():
    pts, w, box, r_min, r_max, _ = small_cfg(51, n=500, L=10.0, r_min=0.5, r_max=2.9)
    nb = 8
    fine = oracle.Graph(pts, None, box, r_min, r_max, nb)
    coarse = oracle.Graph(pts, None, box, r_min, r_max, nb // 2)
    c2f, _ = fine.pcf2()
    c2c, _ = coarse.pcf2()
    assert np.array_equal(c2f.reshape(-1, 2).sum(axis=1), c2c)
    c3f, _ = fine.pcf3()
    c3c, _ = coarse.pcf3()
    folded = np.zeros((nb // 2,) * 3, dtype=np.int64)
    for a, b, c in itertools.product(range(nb), repeat=3):
        v = c3f[(a * nb + b) * nb + c]
        if v:
            folded[tuple(sorted((a // 2, b // 2, c // 2)))] += v
    assert np.array_equal(folded.ravel(), c3c)


# ------------------------------------------------------------------------------------------
# C-6: Poisson closed forms in a periodic box (the paper's analytic-expectation style)

def test_c6_poisson_closed_forms():
    n, L, r_max, nb = 2000, 100.0, 20.0, 10
    V = L ** 3
    e = np.arange(nb + 1) * r_max / nb
    seeds = range(1001, 1013)
    c2 = np.zeros(nb)
    c3 = np.zeros(nb ** 3)
    for s in seeds:
        cfg = catalogues.config1(seed=s)
        g = oracle.Graph(cfg["points"], None, cfg["box"], 0.0, r_max, nb)
        c2 += g.pcf2()[0]
        c3 += g.pcf3()[0]
    k = len(seeds)
    pairs = n * (n - 1) / 2
    exp2 = k * pairs * (4 * math.pi / 3) * (e[1:] ** 3 - e[:-1] ** 3) / V
    # pair counts: relative shot noise ~ 1/sqrt(count)
    assert np.all(np.abs(c2 - exp2) < 5 * np.sqrt(exp2) + 1)
    trip = n * (n - 1) * (n - 2) / 6
    exp_total = k * trip * (5 * math.pi ** 2 / 6) * r_max ** 6 / V ** 2     # <=> 15/32 of neighbour pairs linked
    assert abs(c3.sum() / exp_total - 1) < 0.01
    # per-configuration expectation where the three bins satisfy the triangle inequality everywhere
    checked = 0
    for a, b, c in itertools.combinations_with_replacement(range(nb), 3):
        if e[c + 1] > e[a] + e[b]:
            continue
        mu = {1: 1, 2: 3, 3: 6}[len({a, b, c})]
        expect = k * trip / V ** 2 * mu * 8 * math.pi ** 2 * np.prod([(e[x + 1] ** 2 - e[x] ** 2) / 2 for x in (a, b, c)])
        got = c3[(a * nb + b) * nb + c]
        if expect > 2000:
            assert abs(got / expect - 1) < 6 / math.sqrt(expect) + 0.01, (a, b, c, got, expect)
            checked += 1
    assert checked > 30
    # DDD/RRR -> 1: two independent uniform catalogues give the same histogram within shot noise
    ra = oracle.Graph(catalogues.config1(seed=7)["points"], None, [L] * 3, 0.0, r_max, nb).pcf3()[0]
    rb = oracle.Graph(catalogues.config1(seed=8)["points"], None, [L] * 3, 0.0, r_max, nb).pcf3()[0]
    big = (ra + rb) > 4000
    assert big.sum() > 20 and np.all(np.abs(ra[big] / rb[big] - 1) < 0.15)


def test_c6_four_clique_density():
    # P(three neighbours of a hub are mutually linked) = 0.1582 +- 0.0002 (SURVEY Monte Carlo)
    cfg = catalogues.config3(seed=3001, n=6000, L=500.0 * (6000 / 200000) ** (1 / 3))
    g = oracle.Graph(cfg["points"], None, cfg["box"], 0.0, cfg["r_max"], cfg["nbins"])
    m = 2 * g.n_edges / g.n
    k4 = g.pcf4()[0].sum()
    n = g.n
    v_ratio = (4 * math.pi / 3) * cfg["r_max"] ** 3 / float(np.prod(cfg["box"]))
    expect = n * (n - 1) * (n - 2) * (n - 3) / 24 * v_ratio ** 3 * 0.1582
    assert abs(m / ((n - 1) * v_ratio) - 1) < 0.02
    assert abs(k4 / expect - 1) < 0.06


# ------------------------------------------------------------------------------------------
# C-7 / C-8: isolated rigid units (regression ideas of P:257, injection of P:261)

def _tetra_from_lengths(l01, l02, l03, l12, l13, l23):
    """Vertex coordinates of a tetrahedron with the given edge lengths (v3 on the +z side)."""
    v0 = np.zeros(3)
    v1 = np.array([l01, 0.0, 0.0])
    x2 = (l01 ** 2 + l02 ** 2 - l12 ** 2) / (2 * l01)
    y2 = math.sqrt(l02 ** 2 - x2 ** 2)
    v2 = np.array([x2, y2, 0.0])
    x3 = (l01 ** 2 + l03 ** 2 - l13 ** 2) / (2 * l01)
    y3 = (l02 ** 2 + l03 ** 2 - l23 ** 2 - 2 * x2 * x3) / (2 * y2)
    z3sq = l03 ** 2 - x3 ** 2 - y3 ** 2
    assert z3sq > 0.5, "tetrahedron not embeddable / too flat"
    return np.stack([v0, v1, v2, np.array([x3, y3, math.sqrt(z3sq)])])


def test_c7_isolated_pairs_and_regular_tetrahedra():
    K, r_min, r_max, nb = 60, 1.0, 7.0, 6                    # bins of width 1
    pair = np.array([[0.0, 0.0, 0.0], [3.5, 0.0, 0.0]])      # bin 2
    pts, _, _ = catalogues.isolated_units(pair, K, spacing=20.0, seed=71)
    g = oracle.Graph(pts, None, None, r_min, r_max, nb)
    c2, _ = g.pcf2()
    assert c2.tolist() == [0, 0, K, 0, 0, 0]
    assert g.pcf3()[0].sum() == 0 and g.pcf4()[0].sum() == 0
    s = 4.5                                                   # bin 3
    reg = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=float) * s / (2 * math.sqrt(2))
    pts, _, _ = catalogues.isolated_units(reg, K, spacing=25.0, seed=72)
    w = np.full(len(pts), 2.0)
    g = oracle.Graph(pts, w, None, r_min, r_max, nb)
    c2, w2 = g.pcf2()
    c3, w3 = g.pcf3()
    ec, ew, oc, ow = g.pcf4(parity=True)
    assert c2.tolist() == [0, 0, 0, 6 * K, 0, 0] and w2[3] == 4.0 * 6 * K
    assert c3[(3 * nb + 3) * nb + 3] == 4 * K and c3.sum() == 4 * K and w3.sum() == 8.0 * 4 * K
    i6 = np.ravel_multi_index((3,) * 6, (nb,) * 6)
    assert ec[i6] == K and ec.sum() == K and ew[i6] == 16.0 * K
    assert not oc.any() and not ow.any()                      # achiral configuration: odd == 0 (A-10)
    # connected 4pCF idea (Eq. 4/5): xi only in bin 3 -> zeta_disc = 3 xi^2 at (3,3,3,3,3,3)
    xi = np.zeros(nb)
    xi[3] = 0.7
    zd = oracle.zeta_disc(xi)
    assert abs(zd[i6] - 3 * 0.49) < 1e-12
    # non-zero exactly where at least one pair of opposite edges is (3,3)
    t = np.indices((nb,) * 6).reshape(6, -1)
    opp = ((t[0] == 3) & (t[5] == 3)) | ((t[1] == 3) & (t[4] == 3)) | ((t[2] == 3) & (t[3] == 3))
    assert np.array_equal(zd != 0, opp)


SCALENE = (4.5, 5.5, 6.5, 7.5, 8.5, 9.5)     # l01 < l02 < l03 < l12 < l13 < l23: six different bins


def test_c7_scalene_faces():
    K, r_min, r_max, nb = 40, 4.0, 10.0, 6
    tet = _tetra_from_lengths(*SCALENE)
    pts, _, _ = catalogues.isolated_units(tet, K, spacing=40.0, seed=73)
    g = oracle.Graph(pts, None, None, r_min, r_max, nb)
    c2, _ = g.pcf2()
    assert c2.tolist() == [K] * 6
    c3, _ = g.pcf3()
    faces = [(0, 1, 3), (0, 2, 4), (1, 2, 5), (3, 4, 5)]      # bins of faces 012, 013, 023, 123
    for a, b, c in faces:
        assert c3[(a * nb + b) * nb + c] == K
    assert c3.sum() == 4 * K
    ec, _ = g.pcf4()
    assert ec[np.ravel_multi_index((0, 1, 2, 3, 4, 5), (nb,) * 6)] == K and ec.sum() == K


def test_c8_parity_injection():
    """N_L left + N_R right copies of one scalene tetrahedron: even = N_L + N_R, odd = +-(N_L - N_R)
    at the injected configuration, 0 elsewhere.  With vertices 0..3 in canonical order
    (identity is the unique minimising order for bins 0<1<2<3<4<5) V_true > 0 for the unmirrored
    unit, so the A-11 convention gives +1 per unmirrored and -1 per mirrored unit."""
    r_min, r_max, nb = 4.0, 10.0, 6
    tet = _tetra_from_lengths(*SCALENE)
    v = tet - tet[0]
    assert np.dot(np.cross(v[1], v[2]), v[3]) > 0
    assert oracle.canon4((0, 1, 2, 3, 4, 5)) == ((0, 1, 2, 3, 4, 5), 1)
    i6 = np.ravel_multi_index((0, 1, 2, 3, 4, 5), (nb,) * 6)
    K = 500
    for frac_left, seed in [(1.0, 81), (0.75, 82), (0.5, 83), (0.0, 84)]:
        n_left = int(round(frac_left * K))
        mirror = np.zeros(K, dtype=bool)
        mirror[n_left:] = True                               # "left" := unmirrored
        pts, uid, vid = catalogues.isolated_units(tet, K, spacing=40.0, seed=seed, mirror_mask=mirror)
        g = oracle.Graph(pts, None, None, r_min, r_max, nb)
        ec, ew, oc, ow = g.pcf4(parity=True)
        assert ec[i6] == K and ec.sum() == K
        others = np.delete(oc, i6)
        assert not others.any()
        want = n_left - (K - n_left)
        # pixelised directions (12.7 deg pixels) flip or zero a few per cent of the units at most
        assert abs(oc[i6] - want) <= 0.04 * K, (oc[i6], want)
        if frac_left == 0.5:
            assert abs(oc[i6]) <= 0.04 * K
    # exact version: fixed orientation whose three pixelised spokes are far from coplanar for
    # every choice of hub; translations + random labels only -> every unit contributes exactly +-1
    rng = np.random.default_rng(85)
    K = 64
    rot = catalogues._random_rotations(1, np.random.default_rng(2))[0]
    unit = (tet - tet.mean(axis=0)) @ rot.T
    tab = bn.pixel_table()
    for hub in range(4):                                      # robustly chiral after pixelisation?
        sp_ = [unit[k] - unit[hub] for k in range(4) if k != hub]
        nn = [tab[bn.pixel_of(s[None, :])[0]] for s in sp_]
        exact = np.dot(np.cross(sp_[0], sp_[1]), sp_[2]) / np.prod([np.linalg.norm(s) for s in sp_])
        pixd = np.dot(np.cross(nn[0], nn[1]), nn[2])
        assert abs(pixd) > 0.05 and np.sign(pixd) == np.sign(exact)
    mirror = rng.random(K) < 0.3
    pts = []
    for k in range(K):
        u = unit.copy()
        if mirror[k]:
            u = -u                                            # point inversion = mirror + rotation
        pts.append(u[rng.permutation(4)] + np.array([40.0 * (k % 4), 40.0 * ((k // 4) % 4), 40.0 * (k // 16)]) + 20)
    pts = np.concatenate(pts)
    pts = pts[rng.permutation(len(pts))]
    g = oracle.Graph(pts, None, None, r_min, r_max, nb)
    ec, ew, oc, ow = g.pcf4(parity=True)
    assert ec[i6] == K and oc[i6] == int((~mirror).sum()) - int(mirror.sum())


# ------------------------------------------------------------------------------------------
# C-9: null on a Poisson field; achiral configurations identically zero; degenerate fraction

def test_c9_poisson_null_and_achiral_zero():
    cfg = catalogues.config3(seed=9, n=5000, L=500.0 * (5000 / 200000) ** (1 / 3))
    nb = 4
    g = oracle.Graph(cfg["points"], None, cfg["box"], 0.0, cfg["r_max"], nb)
    ec, _, oc, _ = g.pcf4(parity=True)
    assert ec.sum() > 20000
    n, cfgs = oracle.num_configs(4, nb, want_list=True)
    chiral = 0
    for c in cfgs:
        i6 = np.ravel_multi_index(tuple(c), (nb,) * 6)
        canon, chi = oracle.canon4(c)
        assert canon == tuple(c)
        if chi == 0:
            assert oc[i6] == 0
        else:
            chiral += 1
            assert abs(oc[i6]) <= 5 * math.sqrt(ec[i6]) + 5
    assert n == 276 and chiral == 140                          # SURVEY A-10: 140 of 276 chiral-capable
    assert abs(oc.sum()) <= 5 * math.sqrt(ec.sum())


# ------------------------------------------------------------------------------------------
# C-10: constant power-of-two weights are exact

def test_c10_power_of_two_weights():
    pts, _, box, r_min, r_max, nb = small_cfg(101, n=300, L=9.0, r_max=2.7, nb=4)
    g1 = oracle.Graph(pts, None, box, r_min, r_max, nb)
    g2 = oracle.Graph(pts, np.full(len(pts), 4.0), box, r_min, r_max, nb)
    c3, _ = g1.pcf3()
    _, w3 = g2.pcf3()
    assert np.array_equal(w3, 64.0 * c3)
    ec, _ = g1.pcf4()
    _, ew = g2.pcf4()
    assert np.array_equal(ew, 256.0 * ec)
    c2, _ = g1.pcf2()
    _, w2 = g2.pcf2()
    assert np.array_equal(w2, 16.0 * c2)


# ------------------------------------------------------------------------------------------
# C-11: the configuration counts the paper prints (tests/golden/paper_configuration_counts.txt)

def _cayley_menger(d):
    m = np.ones((5, 5))
    m[0, 0] = 0
    m[1:, 1:] = d ** 2
    return np.linalg.det(m)


def test_c11_paper_configuration_counts():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "paper_configuration_counts.txt")) if l.strip() and l[0] != "#"]
    seen = 0
    for r in rows:
        if r[0] in ("3", "4"):
            assert oracle.num_configs(int(r[0]), int(r[1])) == int(r[2])
            seen += 1
        elif r[0] == "cm":
            nb, want = int(r[1]), int(r[2])
            centres = 20.0 + (np.arange(nb) + 0.5) * (65.0 - 20.0) / nb
            n, cfgs = oracle.num_configs(4, nb, want_list=True)
            ok = 0
            for c in cfgs:
                d = np.zeros((4, 4))
                for (a, b), v in zip([(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)], c):
                    d[a, b] = d[b, a] = centres[v]
                ok += _cayley_menger(d) > 0
            assert ok == want
            seen += 1
    assert seen == 4
    assert oracle.num_configs(3, 18) == math.comb(20, 3) == 1140
    assert oracle.num_configs(4, 6) == 2451 and oracle.num_configs(4, 8) == 12496
    # orbit counting (Burnside over S4 acting on the 6 edges) gives the same numbers
    def burnside(nb):
        return (nb ** 6 + 9 * nb ** 4 + 8 * nb ** 2 + 6 * nb ** 2) // 24   # id, 6+3 with x1^2 x2^2, 8 three-cycles x3^2, 6 four-cycles x2 x4
    for nb in (4, 6, 8):
        assert oracle.num_configs(4, nb) == burnside(nb)


def test_canon4_matches_independent_enumeration():
    rng = np.random.default_rng(3)
    for _ in range(300):
        t = tuple(int(v) for v in rng.integers(0, 4, size=6))
        assert oracle.canon4(t) == bn.canon4(t)


# ------------------------------------------------------------------------------------------
# C-12: Eq. 4 is S4-invariant; Poisson => xi ~ 0

def test_c12_zeta_disc_invariance_and_poisson():
    nb = 4
    xi = np.array([0.9, -0.2, 0.35, 0.1])
    zd = oracle.zeta_disc(xi).reshape((nb,) * 6)
    rng = np.random.default_rng(4)
    pairs = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    for _ in range(50):
        t = tuple(int(v) for v in rng.integers(0, nb, size=6))
        m = {}
        for (a, b), v in zip(pairs, t):
            m[(a, b)] = m[(b, a)] = v
        for p in itertools.permutations(range(4)):
            u = tuple(m[(p[a], p[b])] for a, b in pairs)
            assert abs(zd[u] - zd[t]) < 1e-15
    cfg = catalogues.config1(seed=1001)
    g = oracle.Graph(cfg["points"], None, cfg["box"], 0.0, 20.0, 10)
    xi = oracle.xi_periodic(g.pcf2()[0], g.n, cfg["box"], 0.0, 20.0)
    assert np.all(np.abs(xi[3:]) < 0.05)


# ------------------------------------------------------------------------------------------
# hub filter and the on-demand ("direct") sampled-hub walk

def test_hub_filter_partitions_the_result():
    pts, w, box, r_min, r_max, nb = small_cfg(61, n=500, L=10.0, r_max=2.6, nb=4)
    g = oracle.Graph(pts, w, box, r_min, r_max, nb)
    c3, w3 = g.pcf3()
    parts = [g.pcf3(hubs=(0, g.n, 3)), g.pcf3(hubs=(1, g.n, 3)), g.pcf3(hubs=(2, g.n, 3))]
    assert np.array_equal(sum(p[0] for p in parts), c3)
    assert np.allclose(sum(p[1] for p in parts), w3, rtol=1e-12)
    e, _, o, _ = g.pcf4(parity=True)
    ea, _, oa, _ = g.pcf4(parity=True, hubs=(0, 250, 1))
    eb, _, ob, _ = g.pcf4(parity=True, hubs=(250, g.n, 1))
    assert np.array_equal(ea + eb, e) and np.array_equal(oa + ob, o)
    hubs = np.arange(7, g.n, 50)
    cd, wd = oracle.Graph(pts, w, box, r_min, r_max, nb, lists=False).pcf3_direct(hubs)
    cf, wf = g.pcf3(hubs=(7, g.n, 50))
    assert np.array_equal(cd, cf) and np.allclose(wd, wf, rtol=1e-12)
