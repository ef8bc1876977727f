"""Spherical K-means patching: unit vectors, angular distance, centroid = renormalised mean.

Details the paper leaves open follow SURVEY.md 8(c) R15 / BASELINE.json: 10 Lloyd iterations; full-sky
centroids seeded uniformly on the sphere, region centroids seeded as distinct random pixels of the region;
assignment = largest dot product in fp64, ties to the lowest id; an empty cluster keeps its centroid and
its label (labels are never compacted).  K larger than the number of pixels: one patch per pixel
(PAPER.md:L299).  This is input generation, not part of parity.
"""
import numpy as np


def _assign(vecs: np.ndarray, cent: np.ndarray, chunk: int = 16384) -> np.ndarray:
    out = np.empty(vecs.shape[0], dtype=np.int32)
    ct = np.ascontiguousarray(cent.T)
    for s in range(0, vecs.shape[0], chunk):
        out[s:s + chunk] = np.argmax(vecs[s:s + chunk] @ ct, axis=1)
    return out


def spherical_kmeans(vecs: np.ndarray, K: int, rng: np.random.Generator, iters: int = 10,
                     seed_from_pixels: bool = False) -> np.ndarray:
    """Labels in [0, K_eff) for the rows of `vecs` ([n,3] unit vectors); K_eff = min(K, n)."""
    n = vecs.shape[0]
    if K >= n:
        return np.arange(n, dtype=np.int32)
    if K == 1:
        return np.zeros(n, dtype=np.int32)
    if seed_from_pixels:
        cent = vecs[rng.choice(n, size=K, replace=False)].copy()
    else:
        g = rng.standard_normal((K, 3))
        cent = g / np.linalg.norm(g, axis=1, keepdims=True)
    lab = _assign(vecs, cent)
    for _ in range(iters):
        sums = np.zeros((K, 3))
        np.add.at(sums, lab, vecs)
        nrm = np.linalg.norm(sums, axis=1)
        upd = nrm > 0
        cent[upd] = sums[upd] / nrm[upd, None]
        lab = _assign(vecs, cent)
    return lab
