"""Host-side post-processing above the hot path (S:8(f) rank 1; sec. 3.3): NumPy arithmetic on
the histograms the CUDA library returns.  Nothing here enumerates tuples.

* :func:`xi_periodic`      -- 2pCF of a periodic box without randoms (reading A-12, mode b)
* :func:`zeta3_ratio`      -- zeta = NNN / RRR per configuration from a (weighted) data and a random 3pCF
* :func:`zeta4_connected`  -- Eq. 5: zeta_conn = zeta - zeta_disc, zeta_disc from Eq. 4 (``gramsci_zeta_disc``)
* :func:`combined_catalogue` / :func:`signed_ratio` -- the Szapudi-Szalay form: data and randoms in ONE
  catalogue with weights summing to +1 and -1, so that the weighted k-point sum over a bin is the expansion of
  (D - R)^k (DD - 2DR + RR, ...); the estimate is that sum over the randoms-only sum of the same graph geometry
"""
from __future__ import annotations

import numpy as np


def bin_edges(r_min: float, r_max: float, nbins: int) -> np.ndarray:
    return r_min + np.arange(nbins + 1) * (r_max - r_min) / nbins


def xi_periodic(cnt2: np.ndarray, n: int, box, r_min: float, r_max: float) -> np.ndarray:
    """xi_b = cnt2_b / [C(N,2) (4 pi/3)(e_{b+1}^3 - e_b^3)/V] - 1 for a periodic box (A-12 b)."""
    e = bin_edges(r_min, r_max, cnt2.size)
    rr = 0.5 * n * (n - 1) * (4.0 * np.pi / 3.0) * (e[1:] ** 3 - e[:-1] ** 3) / float(np.prod(box))
    return np.asarray(cnt2, dtype=np.float64) / rr - 1.0


def zeta3_ratio(data_hist: np.ndarray, data_norm: float, rand_hist: np.ndarray, rand_norm: float) -> np.ndarray:
    """NNN/RRR per bin: (data_hist / data_norm^3) / (rand_hist / rand_norm^3); data_norm = sum of the data
    weights (or N for unit weights), rand_norm likewise.  Bins with an empty random histogram give NaN."""
    num = np.asarray(data_hist, dtype=np.float64) / float(data_norm) ** 3
    den = np.asarray(rand_hist, dtype=np.float64) / float(rand_norm) ** 3
    out = np.full(num.shape, np.nan)
    np.divide(num, den, out=out, where=den != 0)
    return out


def equilateral3(hist3: np.ndarray, nbins: int) -> np.ndarray:
    """The equilateral 3pCF (P:135 names it as a separate kernel): the diagonal b1 = b2 = b3 of the dense histogram."""
    h = np.asarray(hist3).reshape(nbins, nbins, nbins)
    return np.array([h[b, b, b] for b in range(nbins)])


def zeta4_connected(zeta4: np.ndarray, xi: np.ndarray) -> np.ndarray:
    """Eq. 5: zeta_conn = zeta - zeta_disc on the dense [nb^6] layout, zeta_disc from Eq. 4 through
    the library's host helper.  Applies to the even channel only."""
    from . import gramsci_zeta_disc
    return np.asarray(zeta4, dtype=np.float64) - gramsci_zeta_disc(np.asarray(xi, dtype=np.float64))


def combined_catalogue(data: np.ndarray, randoms: np.ndarray, w_data=None, w_rand=None):
    """Points and signed, normalised weights of the combined catalogue: data weights sum to +1, random
    weights to -1.  Returns (points [N_D + N_R, 3], weights [N_D + N_R], weights of the randoms alone, sum to +1)."""
    wd = np.ones(data.shape[0]) if w_data is None else np.asarray(w_data, dtype=np.float64)
    wr = np.ones(randoms.shape[0]) if w_rand is None else np.asarray(w_rand, dtype=np.float64)
    wd = wd / wd.sum()
    wr = wr / wr.sum()
    pts = np.ascontiguousarray(np.concatenate([data, randoms], axis=0))
    return pts, np.concatenate([wd, -wr]), wr


def signed_ratio(n_hist: np.ndarray, r_hist: np.ndarray) -> np.ndarray:
    """N...N / R...R per bin (P:118 for pairs; the same form for triplets and quadruplets): n_hist = weighted sums of the
    combined signed catalogue, r_hist = weighted sums of the randoms alone (weights summing to +1).  NaN where the
    random sum is empty."""
    num = np.asarray(n_hist, dtype=np.float64)
    den = np.asarray(r_hist, dtype=np.float64)
    out = np.full(num.shape, np.nan)
    np.divide(num, den, out=out, where=den != 0)
    return out
