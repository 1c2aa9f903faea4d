"""Seeded synthetic point catalogues (inputs only -- none of the method's arithmetic).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2607_06604_b200/``); it imports neither.  Every generator is a pure
function of its seed (``numpy.random.default_rng``, PCG64) and returns host
fp64 arrays.  Recipes follow SURVEY.md section 8(d) / BASELINE.json ``configs``;
they stand in for the catalogues the paper measures on (Gaussian mock, DESI DR1
LRG, Quijote halos), none of which is in this container.

Each ``config_*`` function returns a dict:
    points   float64 [N,3]   (inside [0,L) per axis when periodic)
    weights  float64 [N] or None (None == unit weights)
    box      float64 [3] or None (None == open, non-periodic)
    r_min, r_max, nbins
    kind     "3pcf" | "4pcf" | "4pcf_parity"
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "uniform_box", "neyman_scott", "survey_wedge", "snap",
    "config1", "config2_data", "config2_randoms", "config3", "config4", "config5",
    "isolated_units", "tetra_from_lengths", "SCALENE_EDGES", "CONFIGS",
]


def snap(points: np.ndarray, bits: int = 10) -> np.ndarray:
    """Snap coordinates to a 2**-bits grid so squared distances are exact in fp64."""
    s = float(1 << bits)
    return np.floor(points * s) / s


def uniform_box(n: int, L: float, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.random((n, 3)) * L


def neyman_scott(n: int, L: float, mean_parents: float, sigma: float, seed: int) -> np.ndarray:
    """Neyman-Scott cluster process: Poisson(mean_parents) parents uniform in the box;
    each of the n children picks a parent uniformly and is offset N(0, sigma^2) per axis,
    wrapped periodically."""
    rng = np.random.default_rng(seed)
    n_par = max(1, int(rng.poisson(mean_parents)))
    parents = rng.random((n_par, 3)) * L
    which = rng.integers(0, n_par, size=n)
    pts = parents[which] + rng.normal(0.0, sigma, size=(n, 3))
    pts = np.mod(pts, L)
    pts[pts >= L] = 0.0          # guard against mod() rounding up to L
    return pts


def survey_wedge(n: int, seed: int, ra_deg=(0.0, 30.0), dec_deg=(-15.0, 15.0),
                 r_lo: float = 600.0, r_hi: float = 1400.0,
                 r0: float = 1000.0, sig: float = 200.0) -> np.ndarray:
    """Non-periodic survey-like wedge: RA ~ U, sin(Dec) ~ U, comoving radius with
    pdf proportional to r^2 exp(-(r-r0)^2 / (2 sig^2)) on [r_lo, r_hi] (rejection sampling),
    i.e. number density n(r) proportional to a Gaussian selection."""
    rng = np.random.default_rng(seed)
    ra = np.deg2rad(rng.uniform(ra_deg[0], ra_deg[1], size=n))
    sin_dec = rng.uniform(np.sin(np.deg2rad(dec_deg[0])), np.sin(np.deg2rad(dec_deg[1])), size=n)
    cos_dec = np.sqrt(1.0 - sin_dec * sin_dec)
    # rejection sampling for the radius
    rr = np.linspace(r_lo, r_hi, 4001)
    fmax = float(np.max(rr * rr * np.exp(-0.5 * ((rr - r0) / sig) ** 2))) * 1.001
    out = np.empty(n)
    filled = 0
    while filled < n:
        m = max(1024, 2 * (n - filled))
        cand = rng.uniform(r_lo, r_hi, size=m)
        f = cand * cand * np.exp(-0.5 * ((cand - r0) / sig) ** 2)
        keep = cand[rng.uniform(0.0, fmax, size=m) < f]
        k = min(keep.size, n - filled)
        out[filled:filled + k] = keep[:k]
        filled += k
    x = out * cos_dec * np.cos(ra)
    y = out * cos_dec * np.sin(ra)
    z = out * sin_dec
    return np.stack([x, y, z], axis=1)


def _cfg(points, weights, box, r_min, r_max, nbins, kind, name):
    return dict(points=np.ascontiguousarray(points, dtype=np.float64),
                weights=None if weights is None else np.ascontiguousarray(weights, dtype=np.float64),
                box=None if box is None else np.asarray(box, dtype=np.float64),
                r_min=float(r_min), r_max=float(r_max), nbins=int(nbins), kind=kind, name=name)


def config1(seed: int = 1001, n: int = 2000, L: float = 100.0):
    """BASELINE.json configs[0]: 3pCF, 2000 uniform points, periodic L=100, r<20, 10 bins, unit weights."""
    return _cfg(uniform_box(n, L, seed), None, [L, L, L], 0.0, 20.0, 10, "3pcf", "cfg1")


def config2_data(seed: int = 2001, n: int = 1_000_000, L: float = 1000.0,
                 mean_parents: float = 1.0e4, sigma: float = 5.0):
    """configs[1] data: 1e6 Neyman-Scott points, periodic L=1000, r<30, 15 bins, w ~ U(0.5,1.5).
    Scale n, L^3 and mean_parents together to keep the densities (used by the scaled replicas)."""
    pts = neyman_scott(n, L, mean_parents, sigma, seed)
    w = np.random.default_rng(seed + 500).uniform(0.5, 1.5, size=n)
    return _cfg(pts, w, [L, L, L], 0.0, 30.0, 15, "3pcf", "cfg2D")


def config2_randoms(seed: int = 2002, n: int = 1_000_000, L: float = 1000.0):
    """configs[1] randoms: equal-size uniform catalogue in the same box, unit weights."""
    return _cfg(uniform_box(n, L, seed), None, [L, L, L], 0.0, 30.0, 15, "3pcf", "cfg2R")


def config3(seed: int = 3001, n: int = 200_000, L: float = 500.0):
    """configs[2]: 4pCF, 2e5 uniform points, periodic L=500, r<25, 6 bins, unit weights."""
    return _cfg(uniform_box(n, L, seed), None, [L, L, L], 0.0, 25.0, 6, "4pcf", "cfg3")


def config4(seed: int = 4001, n: int = 500_000, cap_deg: float = 30.0):
    """configs[3]: parity 4pCF, survey wedge (RA x Dec cap cap_deg x cap_deg, r in [600,1400],
    n(r) ~ Gaussian(1000, 200)), open box, r<40, 8 bins, w ~ U(0.8,1.2).
    The scaled replica cfg4' uses n=62_500, cap_deg=15 (same density, ~1/8 of the tuples)."""
    pts = survey_wedge(n, seed, ra_deg=(0.0, cap_deg), dec_deg=(-cap_deg / 2, cap_deg / 2))
    w = np.random.default_rng(seed + 500).uniform(0.8, 1.2, size=n)
    return _cfg(pts, w, None, 0.0, 40.0, 8, "4pcf_parity", "cfg4")


def config5(seed: int = 5001, n: int = 2_500_000, L: float = 1700.0):
    """configs[4]: BAO-scale 3pCF, 2.5e6 uniform points, periodic L=1700, 60<=r<150, 18 bins.
    The scaled replica cfg5' uses L=425, n=39_062 (same density)."""
    return _cfg(uniform_box(n, L, seed), None, [L, L, L], 60.0, 150.0, 18, "3pcf", "cfg5")


SCALENE_EDGES = (4.5, 5.5, 6.5, 7.5, 8.5, 9.5)   # l01 < l02 < l03 < l12 < l13 < l23


def tetra_from_lengths(l01, l02, l03, l12, l13, l23) -> np.ndarray:
    """Vertex coordinates [4,3] of a tetrahedron with the given edge lengths (v3 on the +z side)."""
    x2 = (l01 ** 2 + l02 ** 2 - l12 ** 2) / (2 * l01)
    y2 = float(np.sqrt(l02 ** 2 - x2 ** 2))
    x3 = (l01 ** 2 + l03 ** 2 - l13 ** 2) / (2 * l01)
    y3 = (l02 ** 2 + l03 ** 2 - l23 ** 2 - 2 * x2 * x3) / (2 * y2)
    z3sq = l03 ** 2 - x3 ** 2 - y3 ** 2
    assert z3sq > 0.5, "tetrahedron not embeddable / too flat"
    return np.array([[0.0, 0.0, 0.0], [l01, 0.0, 0.0], [x2, y2, 0.0], [x3, y3, float(np.sqrt(z3sq))]])


def _random_rotations(k: int, rng) -> np.ndarray:
    """k uniformly random proper rotations (QR of Gaussian matrices, det fixed to +1)."""
    a = rng.normal(size=(k, 3, 3))
    q, r = np.linalg.qr(a)
    d = np.sign(np.einsum("kii->ki", r))
    q = q * d[:, None, :]
    det = np.linalg.det(q)
    q[:, :, 0] *= det[:, None]
    return q


def isolated_units(unit: np.ndarray, k: int, spacing: float, seed: int,
                   mirror_mask: np.ndarray | None = None, shuffle: bool = True):
    """k rigid copies of ``unit`` ([n_v,3] vertex coordinates), each randomly rotated and
    placed at a distinct node of a cubic lattice with the given spacing (choose spacing >
    r_max + 2*unit radius so units are mutually isolated); copies flagged in ``mirror_mask``
    are mirrored (x -> -x) before rotation.  Returns (points [k*n_v,3], unit_id [k*n_v],
    vertex_id [k*n_v]) in a random label order (the PAPER.md:257/261 regression / injection idea)."""
    rng = np.random.default_rng(seed)
    nv = unit.shape[0]
    side = int(np.ceil(k ** (1.0 / 3.0)))
    nodes = np.stack(np.meshgrid(*[np.arange(side)] * 3, indexing="ij"), axis=-1).reshape(-1, 3)
    nodes = nodes[rng.permutation(nodes.shape[0])[:k]].astype(np.float64) * spacing
    rot = _random_rotations(k, rng)
    u = np.broadcast_to(unit - unit.mean(axis=0), (k, nv, 3)).copy()
    if mirror_mask is not None:
        u[np.asarray(mirror_mask, dtype=bool), :, 0] *= -1.0
    pts = np.einsum("kij,kvj->kvi", rot, u) + nodes[:, None, :] + spacing  # keep coordinates positive
    pts = pts.reshape(-1, 3)
    uid = np.repeat(np.arange(k), nv)
    vid = np.tile(np.arange(nv), k)
    if shuffle:
        p = rng.permutation(pts.shape[0])
        pts, uid, vid = pts[p], uid[p], vid[p]
    return np.ascontiguousarray(pts), uid, vid


CONFIGS = {
    "cfg1": config1, "cfg2D": config2_data, "cfg2R": config2_randoms,
    "cfg3": config3, "cfg4": config4, "cfg5": config5,
}
