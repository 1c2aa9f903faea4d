"""Independent NumPy statement of the definition (SURVEY.md 8(c) O-def) -- TEST INFRASTRUCTURE.

Written separately from ``gramsci_oracle.c`` and deliberately with *different* formulas where the
mathematics allows it (sqrt + floor binning instead of squared-edge comparisons; ``min(|d|, L-|d|)``
instead of the signed minimum image; ``arctan2`` / floor pixelisation instead of tangent
comparisons; ``itertools.permutations`` canonicalisation), so that a slip in either shows up as
a disagreement on random inputs (the two formulations can only differ when a value lands within
one ulp of a bin / pixel boundary).  O(N^2) memory, O(N^3..N^4) time: tiny N only.
"""
from __future__ import annotations

import itertools

import numpy as np


def adjacency(points, box, r_min, r_max, nbins):
    """Dense bin matrix B [N,N] (int, -1 = no edge) and separation vectors D [N,N,3] (row -> col)."""
    x = np.asarray(points, dtype=np.float64)
    d = x[None, :, :] - x[:, None, :]                     # d[i,j] = x_j - x_i
    if box is not None:
        L = np.asarray(box, dtype=np.float64)
        d = d - L * np.round(d / L)                       # nearest image
    r = np.sqrt((d * d).sum(axis=2))
    width = (r_max - r_min) / nbins
    b = np.floor((r - r_min) / width).astype(np.int64)
    ok = (r >= r_min) & (r < r_max)
    np.fill_diagonal(ok, False)
    b = np.where(ok, np.clip(b, 0, nbins - 1), -1)
    return b, d


def pixel_of(d):
    """256 equal-area pixels: 16 bands in z x 16 sectors in phi (A-8), via arctan2 / floor."""
    r = np.sqrt((d * d).sum(axis=-1))
    r = np.where(r > 0, r, 1.0)
    iz = np.clip(np.floor((d[..., 2] / r + 1.0) * 8.0), 0, 15).astype(np.int64)
    phi = np.mod(np.arctan2(d[..., 1], d[..., 0]), 2.0 * np.pi)
    ip = np.clip(np.floor(phi / (np.pi / 8.0)), 0, 15).astype(np.int64)
    return 16 * iz + ip


def pixel_table():
    p = np.arange(256)
    zc = ((p >> 4) + 0.5) / 8.0 - 1.0
    ph = ((p & 15) + 0.5) * np.pi / 8.0
    s = np.sqrt(1.0 - zc * zc)
    return np.stack([s * np.cos(ph), s * np.sin(ph), zc], axis=1)


_PERMS = list(itertools.permutations(range(4)))


def _perm_sign(p):
    inv = sum(1 for a in range(4) for b in range(a + 1, 4) if p[a] > p[b])
    return -1 if inv & 1 else 1


def canon4(t):
    """Lexicographic minimum of the 6-tuple over the 24 vertex orders, and the chirality factor."""
    m = {}
    pairs = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    for (a, b), v in zip(pairs, t):
        m[(a, b)] = m[(b, a)] = int(v)
    best, signs = None, set()
    for p in _PERMS:
        u = tuple(m[(p[a], p[b])] for a, b in pairs)
        if best is None or u < best:
            best, signs = u, {_perm_sign(p)}
        elif u == best:
            signs.add(_perm_sign(p))
    return best, (0 if len(signs) == 2 else signs.pop())


def pcf2(points, weights, box, r_min, r_max, nbins):
    b, _ = adjacency(points, box, r_min, r_max, nbins)
    w = np.ones(len(points)) if weights is None else np.asarray(weights, dtype=np.float64)
    iu = np.triu_indices(len(points), 1)
    bb = b[iu]
    ok = bb >= 0
    cnt = np.bincount(bb[ok], minlength=nbins).astype(np.int64)
    ws = np.bincount(bb[ok], weights=(w[iu[0]] * w[iu[1]])[ok], minlength=nbins)
    return cnt, ws


def pcf3(points, weights, box, r_min, r_max, nbins):
    b, _ = adjacency(points, box, r_min, r_max, nbins)
    n = len(points)
    w = np.ones(n) if weights is None else np.asarray(weights, dtype=np.float64)
    cnt = np.zeros((nbins,) * 3, dtype=np.int64)
    ws = np.zeros((nbins,) * 3, dtype=np.float64)
    for i in range(n):
        for j in range(i + 1, n):
            if b[i, j] < 0:
                continue
            k = np.nonzero((b[i, j + 1:] >= 0) & (b[j, j + 1:] >= 0))[0] + j + 1
            if k.size == 0:
                continue
            tri = np.sort(np.stack([np.full(k.size, b[i, j]), b[i, k], b[j, k]], axis=1), axis=1)
            np.add.at(cnt, (tri[:, 0], tri[:, 1], tri[:, 2]), 1)
            np.add.at(ws, (tri[:, 0], tri[:, 1], tri[:, 2]), w[i] * w[j] * w[k])
    return cnt.ravel(), ws.ravel()


def pcf4(points, weights, box, r_min, r_max, nbins, parity=False):
    b, d = adjacency(points, box, r_min, r_max, nbins)
    n = len(points)
    w = np.ones(n) if weights is None else np.asarray(weights, dtype=np.float64)
    tab = pixel_table()
    pix = pixel_of(d)
    even_c = np.zeros((nbins,) * 6, dtype=np.int64)
    even_w = np.zeros((nbins,) * 6, dtype=np.float64)
    odd_c = np.zeros((nbins,) * 6, dtype=np.int64)
    odd_w = np.zeros((nbins,) * 6, dtype=np.float64)
    cache = {}
    for i in range(n):
        ni = np.nonzero(b[i, i + 1:] >= 0)[0] + i + 1
        for a, j in enumerate(ni):
            for k in ni[a + 1:]:
                if b[j, k] < 0:
                    continue
                ls = ni[(ni > k)]
                ls = ls[(b[j, ls] >= 0) & (b[k, ls] >= 0)]
                for l in ls:
                    t = (b[i, j], b[i, k], b[i, l], b[j, k], b[j, l], b[k, l])
                    if t not in cache:
                        cache[t] = canon4(t)
                    c, chi = cache[t]
                    ww = w[i] * w[j] * w[k] * w[l]
                    even_c[c] += 1
                    even_w[c] += ww
                    if parity:
                        v = float(np.dot(np.cross(tab[pix[i, j]], tab[pix[i, k]]), tab[pix[i, l]]))
                        s = 0 if abs(v) < 1e-9 else (1 if v > 0 else -1)
                        odd_c[c] += chi * s
                        odd_w[c] += chi * s * ww
    if parity:
        return even_c.ravel(), even_w.ravel(), odd_c.ravel(), odd_w.ravel()
    return even_c.ravel(), even_w.ravel()
