"""CPU oracle for the GRAMSCI hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2607_06604_b200`` and never imports it.  See ``gramsci_oracle.c`` for the
arithmetic (each function cites the PAPER.md passage it follows) and ``brute_numpy.py``
for an independently written NumPy statement of the definition.

The C file is compiled on first use with
``gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gramsci_oracle.c")
_LIB = os.path.join(_HERE, "libgramsci_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = ctypes.CDLL(_LIB)
    c_dp = ctypes.POINTER(ctypes.c_double)
    c_i64p = ctypes.POINTER(ctypes.c_int64)
    L.og_build.restype = ctypes.c_void_p
    L.og_build.argtypes = [c_dp, c_dp, ctypes.c_int64, c_dp, ctypes.c_double, ctypes.c_double,
                           ctypes.c_int, ctypes.c_int, ctypes.c_int]
    L.og_free.argtypes = [ctypes.c_void_p]
    L.og_num_edges.restype = ctypes.c_int64
    L.og_num_edges.argtypes = [ctypes.c_void_p]
    L.og_export.argtypes = [ctypes.c_void_p] + [ctypes.c_void_p] * 4
    L.og_2pcf.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    L.og_3pcf.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p] + [ctypes.c_int64] * 3
    L.og_4pcf.argtypes = [ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 4 + [ctypes.c_int64] * 3
    L.og_brute_2pcf.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    L.og_brute_3pcf.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    L.og_brute_4pcf.argtypes = [ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 4
    L.og_3pcf_direct.argtypes = [ctypes.c_void_p, c_i64p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
    L.og_degrees_direct.argtypes = [ctypes.c_void_p, c_i64p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
    L.og_num_configs.restype = ctypes.c_int64
    L.og_num_configs.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
    L.og_canon4.restype = ctypes.c_int
    L.og_canon4.argtypes = [ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]
    L.og_pixel_centre.argtypes = [ctypes.c_int, c_dp]
    L.og_zeta_disc.argtypes = [ctypes.c_int, c_dp, c_dp]
    L.og_threads.restype = ctypes.c_int
    _lib = L
    return L


def _dp(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _vp(a: Optional[np.ndarray]):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


def threads() -> int:
    return int(_load().og_threads())


class Graph:
    """Radius graph of a catalogue (O-def step 1).  ``lists=False`` keeps only the cell list
    (for the ``*_direct`` sampled-hub functions on graphs too large to hold)."""

    def __init__(self, points, weights=None, box=None, r_min=0.0, r_max=1.0, nbins=1,
                 use_cells=True, lists=True):
        L = _load()
        self.points = np.ascontiguousarray(points, dtype=np.float64)
        assert self.points.ndim == 2 and self.points.shape[1] == 3
        self.weights = None if weights is None else np.ascontiguousarray(weights, dtype=np.float64)
        self.box = None if box is None else np.ascontiguousarray(box, dtype=np.float64)
        self.n = self.points.shape[0]
        self.nb = int(nbins)
        self.r_min, self.r_max = float(r_min), float(r_max)
        self._h = L.og_build(_dp(self.points), _dp(self.weights), self.n, _dp(self.box),
                             self.r_min, self.r_max, self.nb, int(bool(use_cells)), int(bool(lists)))
        if not self._h:
            raise ValueError("oracle: invalid arguments (bins, radii, or r_max >= box/2)")
        self.has_lists = bool(lists)

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.og_free(h)

    # -- graph ---------------------------------------------------------------------------
    @property
    def n_edges(self) -> int:
        return int(_load().og_num_edges(self._h))

    def csr(self):
        """(start int64 [n+1], idx int32 [E], bin uint8 [E], pix uint8 [E]) oriented, sorted rows."""
        E = self.n_edges
        start = np.zeros(self.n + 1, dtype=np.int64)
        idx = np.zeros(max(E, 1), dtype=np.int32)
        b = np.zeros(max(E, 1), dtype=np.uint8)
        p = np.zeros(max(E, 1), dtype=np.uint8)
        _load().og_export(self._h, _vp(start), _vp(idx), _vp(b), _vp(p))
        return start, idx[:E], b[:E], p[:E]

    # -- queries -------------------------------------------------------------------------
    def _hubs(self, hubs):
        hb, he, hs = (0, self.n, 1) if hubs is None else hubs
        return int(hb), int(he), int(hs)

    def pcf2(self, brute=False):
        cnt = np.zeros(self.nb, dtype=np.int64)
        ws = np.zeros(self.nb, dtype=np.float64)
        f = _load().og_brute_2pcf if brute else _load().og_2pcf
        f(self._h, _vp(cnt), _vp(ws))
        return cnt, ws

    def pcf3(self, hubs=None, brute=False):
        nh = self.nb ** 3
        cnt = np.zeros(nh, dtype=np.int64)
        ws = np.zeros(nh, dtype=np.float64)
        if brute:
            _load().og_brute_3pcf(self._h, _vp(cnt), _vp(ws))
        else:
            _load().og_3pcf(self._h, _vp(cnt), _vp(ws), *self._hubs(hubs))
        return cnt, ws

    def pcf4(self, parity=False, hubs=None, brute=False):
        nh = self.nb ** 6
        ec = np.zeros(nh, dtype=np.int64)
        ew = np.zeros(nh, dtype=np.float64)
        oc = np.zeros(nh, dtype=np.int64) if parity else None
        ow = np.zeros(nh, dtype=np.float64) if parity else None
        if brute:
            _load().og_brute_4pcf(self._h, int(parity), _vp(ec), _vp(ew), _vp(oc), _vp(ow))
        else:
            _load().og_4pcf(self._h, int(parity), _vp(ec), _vp(ew), _vp(oc), _vp(ow), *self._hubs(hubs))
        return (ec, ew, oc, ow) if parity else (ec, ew)

    def pcf3_direct(self, hub_labels):
        hubs = np.ascontiguousarray(hub_labels, dtype=np.int64)
        nh = self.nb ** 3
        cnt = np.zeros(nh, dtype=np.int64)
        ws = np.zeros(nh, dtype=np.float64)
        _load().og_3pcf_direct(self._h, hubs.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
                               hubs.size, _vp(cnt), _vp(ws))
        return cnt, ws

    def degrees_direct(self, labels):
        pts = np.ascontiguousarray(labels, dtype=np.int64)
        full = np.zeros(pts.size, dtype=np.int64)
        plus = np.zeros(pts.size, dtype=np.int64)
        _load().og_degrees_direct(self._h, pts.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
                                  pts.size, _vp(full), _vp(plus))
        return full, plus


def num_configs(npoint: int, nbins: int, want_list: bool = False):
    L = _load()
    n = int(L.og_num_configs(npoint, nbins, None))
    if not want_list:
        return n
    cfg = np.zeros((n, 3 if npoint == 3 else 6), dtype=np.int32)
    L.og_num_configs(npoint, nbins, _vp(cfg))
    return n, cfg


def canon4(t):
    """(canonical 6-tuple, chirality factor) of a raw 6-tuple (b01,b02,b03,b12,b13,b23)."""
    a = (ctypes.c_int * 6)(*[int(v) for v in t])
    c = (ctypes.c_int * 6)()
    g = _load().og_canon4(a, c)
    return tuple(int(v) for v in c), int(g)


def pixel_centres() -> np.ndarray:
    tab = np.zeros((256, 3), dtype=np.float64)
    L = _load()
    for p in range(256):
        L.og_pixel_centre(p, _dp(tab[p]))
    return tab


def zeta_disc(xi: np.ndarray) -> np.ndarray:
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    out = np.zeros(xi.size ** 6, dtype=np.float64)
    _load().og_zeta_disc(xi.size, _dp(xi), _dp(out))
    return out


def xi_periodic(cnt2: np.ndarray, n: int, box, r_min: float, r_max: float) -> np.ndarray:
    """S:8(c) A-12 mode (b): xi_b = cnt2_b / [C(N,2) (4 pi/3)(e_{b+1}^3 - e_b^3)/V] - 1."""
    nb = cnt2.size
    e = r_min + np.arange(nb + 1) * (r_max - r_min) / nb
    vol = float(np.prod(box))
    rr = 0.5 * n * (n - 1) * (4.0 * np.pi / 3.0) * (e[1:] ** 3 - e[:-1] ** 3) / vol
    return cnt2 / rr - 1.0
