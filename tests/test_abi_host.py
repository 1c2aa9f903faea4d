"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/gramsci.h declares,
its host-only helpers agree with the paper's printed configuration counts, and compute entry points
fail loudly (GRAMSCI_ECUDA) when no CUDA device is present -- there is no CPU fallback."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2607_06604_b200 as gr
from paper_2607_06604_b200 import build as gr_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    gr_build.build()
    return gr.load_library()


def test_header_symbols_are_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "gramsci.h")).read()
    declared = set(re.findall(r"\b(gramsci_[a-z0-9_]+)\s*\(", hdr))
    declared -= {"gramsci_graph", "gramsci_status", "gramsci_options"}
    assert declared == set(gr.ABI_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_paper_configuration_counts(lib):
    # P:285 (220), P:257 (680), P:291 (276): tests/golden/paper_configuration_counts.txt
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_configuration_counts.txt")):
        f = line.split()
        if not f or f[0] not in ("3", "4"):
            continue
        assert gr.gramsci_num_configs(int(f[0]), int(f[1])) == int(f[2])
    assert gr.gramsci_num_configs(4, 6) == 2451
    assert gr.gramsci_num_configs(4, 8) == 12496


def test_compact_lists_sorted_triples(lib):
    nb = 4
    dense = np.arange(nb ** 3, dtype=np.int64)
    vals, bins = gr.gramsci_compact(3, nb, dense)
    assert len(vals) == 20
    assert all(a <= b <= c for a, b, c in bins)
    assert all(vals[k] == (bins[k][0] * nb + bins[k][1]) * nb + bins[k][2] for k in range(len(vals)))
    vals4, bins4 = gr.gramsci_compact(4, 2, np.arange(64, dtype=np.int64))
    assert len(vals4) == gr.gramsci_num_configs(4, 2) == 11


def test_zeta_disc_is_s4_invariant(lib):
    rng = np.random.default_rng(5)
    nb = 3
    xi = rng.normal(size=nb)
    z = gr.gramsci_zeta_disc(xi).reshape((nb,) * 6)
    # swapping vertices 1 and 2 maps (b12,b13,b14,b23,b24,b34) -> (b12,b23,b24,b13,b14,b34)
    assert np.allclose(z, z.transpose(0, 3, 4, 1, 2, 5))
    t = (0, 1, 2, 2, 1, 0)
    assert np.isclose(z[t], xi[0] * xi[0] + xi[1] * xi[1] + xi[2] * xi[2])


def test_argument_errors(lib):
    pts = np.zeros((4, 3))
    with pytest.raises(gr.GramsciError) as e:
        gr.gramsci_build_graph(pts, None, None, 0.0, 1.0, 0)
    assert e.value.code == 1
    with pytest.raises(gr.GramsciError) as e:
        gr.gramsci_build_graph(pts, None, None, 2.0, 1.0, 4)
    assert e.value.code == 1


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    pts = np.random.default_rng(0).random((10, 3))
    with pytest.raises(gr.GramsciError) as e:
        gr.gramsci_build_graph(pts, None, [1.0, 1.0, 1.0], 0.0, 0.3, 4)
    assert e.value.code == 4          # GRAMSCI_ECUDA
    assert "no CPU fallback" in str(e.value)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2607_06604_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("the oracle", "").replace("oracle's", ""), f


def test_estimator_helpers(lib):
    from paper_2607_06604_b200 import estimators as est
    # a periodic Poisson box has xi = 0 when the pair counts sit on their expectation
    n, box, nb = 1000, [50.0, 50.0, 50.0], 4
    e = est.bin_edges(0.0, 8.0, nb)
    expect = 0.5 * n * (n - 1) * (4 * np.pi / 3) * (e[1:] ** 3 - e[:-1] ** 3) / 50.0 ** 3
    assert np.allclose(est.xi_periodic(expect, n, box, 0.0, 8.0), 0.0)
    # NNN/RRR: doubling every data weight multiplies the histogram by 8 and the norm by 2 -> same zeta
    h = np.arange(1, 9, dtype=np.float64)
    assert np.allclose(est.zeta3_ratio(8 * h, 2 * 10.0, h, 10.0), 1.0)
    assert np.isnan(est.zeta3_ratio(h, 1.0, np.zeros(8), 1.0)).all()
    # Eq. 5 with xi = 0 leaves zeta untouched
    z = np.random.default_rng(1).normal(size=3 ** 6)
    assert np.array_equal(est.zeta4_connected(z, np.zeros(3)), z)
