"""Pins of the K-means reference oracle/kmeans.py (f2; R15) against what the paper
and the mathematics fix, then the input generator gen/kmeans.py (which keeps a faster evaluation) against it.

Each pin is chosen so that a plausible mistake fails it: argmin for argmax, a missing renormalisation, a mean over the
wrong pixels, a wrong tie or empty-patch rule, an assignment that does not follow the last update.
"""
import numpy as np
import pytest

import gen
from gen import kmeans as gk
from gen import sky
from oracle import kmeans as ok


def _random_unit(n, seed):
    g = np.random.default_rng(seed).standard_normal((n, 3))
    return g / np.linalg.norm(g, axis=1, keepdims=True)


def test_assignment_is_the_nearest_centroid_in_angular_distance():
    """L100-L102: a pixel belongs to the centroid at the smallest angle.  Generic points, so no ties."""
    v, c = _random_unit(4000, 1), _random_unit(37, 2)
    lab = ok.assign(v, c)
    ang = np.arccos(np.clip(v @ c.T, -1.0, 1.0))
    assert np.array_equal(lab, np.argmin(ang, axis=1))
    assert lab.dtype == np.int32 and len(np.unique(lab)) == 37


def test_octahedron_closed_form():
    """Centroids at +-x, +-y, +-z: the nearest one is given by the coordinate of largest magnitude and its sign."""
    v = _random_unit(5000, 3)
    c = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], dtype=np.float64)
    axis = np.argmax(np.abs(v), axis=1)
    want = 2 * axis + (v[np.arange(v.shape[0]), axis] < 0)
    assert np.array_equal(ok.assign(v, c), want)


def test_ties_go_to_the_lowest_id():
    v = gen.pix2vec_ring(8)
    a, b = _random_unit(2, 4)
    for cent, never in (([a, b, a], 2), ([b, a, a], 2), ([a, a, b], 1)):
        lab = ok.assign(v, np.array(cent))
        assert not np.any(lab == never) and len(np.unique(lab)) == 2
    # exact ties from the pixel symmetries themselves: poles as centroids, the equatorial ring (z == 0) goes to id 0
    v4 = gen.pix2vec_ring(4)
    ring = v4[:, 2] == 0.0
    assert ring.sum() == 16
    assert np.all(ok.assign(v4, np.array([[0, 0, 1.0], [0, 0, -1.0]]))[ring] == 0)
    assert np.all(ok.assign(v4, np.array([[0, 0, -1.0], [0, 0, 1.0]]))[ring] == 0)


def test_update_is_the_renormalised_mean_and_an_empty_patch_keeps_its_centroid():
    """L104.  Recomputed with np.add.at (ascending pixel order, one add at a time) -- bit for bit -- and against the
    mean itself: normalise(mean) to rounding."""
    v = gen.pix2vec_ring(16)
    c0 = _random_unit(9, 5)
    c0[6] = c0[2]                       # a duplicate of a lower id: patch 6 gets no pixel
    lab = ok.assign(v, c0)
    assert not np.any(lab == 6)
    c1 = ok.update(v, lab, c0)
    assert np.array_equal(c1[6], c0[6])                                  # kept, bit for bit
    sums = np.zeros((9, 3))
    np.add.at(sums, lab, v)
    live = np.arange(9) != 6
    nrm = np.sqrt((sums[:, 0] * sums[:, 0] + sums[:, 1] * sums[:, 1]) + sums[:, 2] * sums[:, 2])
    assert np.array_equal(c1[live], sums[live] / nrm[live, None])
    np.testing.assert_allclose(np.linalg.norm(c1, axis=1), 1.0, rtol=0, atol=4e-16)
    for k in np.flatnonzero(live):
        mean = v[lab == k].mean(axis=0)
        np.testing.assert_allclose(c1[k], mean / np.linalg.norm(mean), rtol=0, atol=1e-14)
    assert not np.allclose(c1[live], c0[live])                           # the update moved them


def test_lloyd_returns_consistent_labels_and_centroids_and_never_lowers_the_objective():
    v = gen.pix2vec_ring(16)
    c0 = _random_unit(40, 6)
    lab, cent, obj = ok.lloyd(v, c0, iters=10, want_objective=True)
    # the labels are the assignment to the centroids that are returned (not to the ones before the last update)
    dots = v @ cent.T
    assert np.all(dots[np.arange(v.shape[0]), lab] >= dots.max(axis=1) - 4e-16)
    assert np.array_equal(lab, ok.assign(v, cent))
    # both Lloyd steps maximise sum_p n_p . c_label(p): it cannot go down, and here it goes up
    assert obj.shape == (11,) and np.all(np.diff(obj) >= -1e-9) and obj[-1] > obj[0] + 1.0
    assert abs(obj[-1] - ok.objective(v, lab, cent)) < 1e-9
    # zero iterations = the first assignment; the iterations are the two steps applied in turn
    lab0, cent0 = ok.lloyd(v, c0, iters=0)
    assert np.array_equal(lab0, ok.assign(v, c0)) and np.array_equal(cent0, c0)
    c, l = c0, lab0
    for _ in range(3):
        c = ok.update(v, l, c)
        l = ok.assign(v, c)
    lab3, cent3 = ok.lloyd(v, c0, iters=3)
    assert np.array_equal(l, lab3) and np.array_equal(c, cent3)
    # relabelling the centroids relabels the patches (no ties among generic centroids)
    perm = np.random.default_rng(7).permutation(40)
    labp, centp = ok.lloyd(v, c0[perm], iters=10)
    assert np.array_equal(perm[labp], lab) and np.array_equal(centp, cent[perm])


def test_antipodal_seeds_split_the_sphere_at_the_equator():
    v = gen.pix2vec_ring(8)
    z = v[:, 2]
    for iters in (0, 1):
        lab, cent = ok.lloyd(v, np.array([[0.0, 0.0, 1.0], [0.0, 0.0, -1.0]]), iters=iters)
        assert np.all(lab[z > 1e-12] == 0) and np.all(lab[z < -1e-12] == 1)
    # the pixel set is symmetric under the quarter turn about z: the open hemispheres' means lie on the axis (the ring at
    # the equator, z = 0 to rounding, is split by the tie rule and tilts them by at most its share of the pixels)
    assert np.all(np.abs(cent[:, :2]) < 32 / 384) and cent[0, 2] > 0.99 and cent[1, 2] < -0.99


def test_fixed_point_on_base_pixel_centres():
    """The 12 nside-1 pixel centres as seeds on the nside-8 pixels: every pixel sits with the centre at the smallest
    angle, and the patch sizes add up; the paper's nearest-centroid rule (L100-L102) with the tie rule of R15."""
    v, seeds = gen.pix2vec_ring(8), gen.pix2vec_ring(1)
    lab, cent = ok.lloyd(v, seeds, iters=0)
    ang = np.arccos(np.clip(v @ seeds.T, -1.0, 1.0))
    assert np.all(ang[np.arange(768), lab] <= ang.min(axis=1) + 1e-12)
    first = np.argmax(ang <= ang.min(axis=1, keepdims=True) + 1e-12, axis=1)   # lowest id among the (near-)tied
    assert np.array_equal(lab, first)
    assert np.bincount(lab, minlength=12).sum() == 768 and np.bincount(lab, minlength=12).min() >= 48


def test_patch_map_rules():
    v = gen.pix2vec_ring(8)
    never = lambda r, sel: pytest.fail("no K-means problem to seed")
    lab, kt = ok.patch_map(v, 5000, never)                                # L299: K > npix
    assert kt == 768 and np.array_equal(lab, np.arange(768))
    lab, kt = ok.patch_map(v, 768, never)
    assert kt == 768 and np.array_equal(lab, np.arange(768))
    lab, kt = ok.patch_map(v, 1, lambda r, sel: v[:1])
    assert kt == 1 and np.all(lab == 0)
    # regions are independent problems whose ids run on (L267): each region's part is the K-means of its pixels alone
    reg = gen.latitude_regions(v)
    seeds = {r: _random_unit(6, 10 + r) for r in range(3)}
    lab, kt = ok.patch_map(v, 6, lambda r, sel: seeds[r], reg, 3)
    assert kt == 18
    for r in range(3):
        sel = np.flatnonzero(reg == r)
        alone, _ = ok.lloyd(v[sel], seeds[r], 10)
        assert np.array_equal(lab[sel], alone + 6 * r)
    # a region smaller than K: one patch per pixel there, K elsewhere
    small = np.zeros(768, dtype=np.uint8)
    small[:4] = 1
    lab, kt = ok.patch_map(v, 6, lambda r, sel: _random_unit(6, 20), small, 2)
    assert kt == 10 and np.array_equal(lab[:4], 6 + np.arange(4)) and lab[4:].max() == 5


def _oracle_map(vecs, param, K, region_idx=None, nregion=1):
    """oracle.kmeans.patch_map on the generator's seeded draws (the random numbers of the method are inputs)."""
    def cent0(r, sel):
        seed = (param * 1_000_003 + K) * 16 + (0 if r is None else r + 1)
        return gk.initial_centroids(vecs[sel], K, sky.rng_for("kmeans", seed), seed_from_pixels=r is not None)
    return ok.patch_map(vecs, K, cent0, region_idx, nregion)


def test_generator_equals_the_reference_on_the_workloads_maps():
    """gen/kmeans.py keeps a faster evaluation (BLAS candidates, exact decision of near ties); its maps -- the inputs of
    every workload -- must be those of the plain reference, bit for bit: C1, C2, the corners and the middle of the C3
    grid, the C4 region maps."""
    v8, v64 = gen.pix2vec_ring(8), gen.pix2vec_ring(64)
    cases = [(v8, p, K, None, 1) for p, K in ((0, 4), (1, 2), (2, 3))]
    cases += [(v64, p, K, None, 1) for p, K in ((0, 500), (1, 50), (2, 100))]
    grid = gen.c3_grid()
    for p in range(3):
        ks = sorted(set(int(k) for k in grid[p]))
        cases += [(v64, p, K, None, 1) for K in (ks[0], ks[len(ks) // 2], ks[-1])]
    reg = gen.latitude_regions(v64)
    cases += [(v64, 0, 200, reg, 3), (v64, 1, 20, reg, 3), (v64, 2, 50, reg, 3)]
    for vecs, p, K, region_idx, nregion in cases:
        want, kt = _oracle_map(vecs, p, K, region_idx, nregion)
        got, kt2 = gen.cluster_map(vecs, p, K, region_idx, nregion)
        assert kt == kt2 and np.array_equal(got, want), (p, K, nregion, int((got != want).sum()))


def test_generator_kmeans_rules():
    """The generator's own entry point against the reference on a small sphere, centroid by centroid."""
    v = gen.pix2vec_ring(8)
    lab = gen.spherical_kmeans(v, 7, gen.rng_for("kmeans", 5))
    c0 = gk.initial_centroids(v, 7, gen.rng_for("kmeans", 5))
    want, cent = ok.lloyd(v, c0, 10)
    assert np.array_equal(lab, want)
    dots = v @ cent.T
    assert np.all(dots[np.arange(768), lab] >= dots.max(axis=1) - 4e-16)   # each pixel sits with its nearest centroid
