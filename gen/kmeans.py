"""Spherical K-means patching: unit vectors, angular distance, centroid = renormalised mean.

Details the paper leaves open follow SURVEY.md 8(c) R15 / BASELINE.json: 10 Lloyd iterations; full-sky
centroids seeded uniformly on the sphere, region centroids seeded as distinct random pixels of the region;
assignment = largest dot product in fp64, ties to the lowest id; an empty cluster keeps its centroid and
its label (labels are never compacted).  K larger than the number of pixels: one patch per pixel
(PAPER.md:L299).  This is input generation, not part of parity.
"""
import numpy as np


def _assign(vecs: np.ndarray, cent: np.ndarray, chunk: int = 16384) -> np.ndarray:
    """argmax_k n_p . c_k, ties to the lowest id, with the dot product DEFINED as (x cx + y cy) + z cz, every operation
    rounded once (no FMA): region problems are seeded from pixel centres, whose symmetries produce exactly tied dot
    products, so the result must not depend on how a library associates the three terms.
    For speed the BLAS product finds the candidates (everything within 1e-12 of the row maximum, far above any
    rounding difference between the two evaluations); only rows with more than one candidate are decided by the
    defining expression, so the labels are exactly those of the definition."""
    out = np.empty(vecs.shape[0], dtype=np.int32)
    ct = np.ascontiguousarray(cent.T)
    cx, cy, cz = (np.ascontiguousarray(cent[:, i])[None, :] for i in range(3))
    for s in range(0, vecs.shape[0], chunk):
        v = vecs[s:s + chunk]
        dots = v @ ct
        lab = np.argmax(dots, axis=1)
        rows = np.arange(v.shape[0])
        best = dots[rows, lab]
        dots[rows, lab] = -np.inf
        close = np.flatnonzero(best - dots.max(axis=1) <= 1e-12)       # a runner-up within 1e-12 of the maximum
        if close.size:
            vc = v[close]
            exact = (vc[:, 0:1] * cx + vc[:, 1:2] * cy) + vc[:, 2:3] * cz
            lab[close] = np.argmax(exact, axis=1)
        out[s:s + chunk] = lab
    return out


def initial_centroids(vecs: np.ndarray, K: int, rng: np.random.Generator, seed_from_pixels: bool = False) -> np.ndarray:
    """The seeded start of a K-means problem ([K,3] fp64): uniform on the sphere, or K distinct random pixels."""
    if seed_from_pixels:
        return vecs[rng.choice(vecs.shape[0], size=K, replace=False)].copy()
    g = rng.standard_normal((K, 3))
    return g / np.linalg.norm(g, axis=1, keepdims=True)


def spherical_kmeans(vecs: np.ndarray, K: int, rng: np.random.Generator, iters: int = 10,
                     seed_from_pixels: bool = False) -> np.ndarray:
    """Labels in [0, K_eff) for the rows of `vecs` ([n,3] unit vectors); K_eff = min(K, n)."""
    n = vecs.shape[0]
    if K >= n:
        return np.arange(n, dtype=np.int32)
    if K == 1:
        return np.zeros(n, dtype=np.int32)
    cent = initial_centroids(vecs, K, rng, seed_from_pixels)
    lab = _assign(vecs, cent)
    for _ in range(iters):
        # sums[k] = sum of the patch's pixels in ascending pixel order, one fp64 add at a time (bincount walks its input
        # in order, like np.add.at, and is much faster)
        sums = np.stack([np.bincount(lab, weights=vecs[:, i], minlength=K) for i in range(3)], axis=1)
        nrm = np.linalg.norm(sums, axis=1)
        upd = nrm > 0
        cent[upd] = sums[upd] / nrm[upd, None]
        lab = _assign(vecs, cent)
    return lab
