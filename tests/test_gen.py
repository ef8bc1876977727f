"""Input generator checks (CPU): HEALPix RING geometry (R16), noise conversion (R6), K-means rules (R15), recipes."""
import os

import numpy as np

import gen

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_healpix_nside1_matches_published_scheme():
    tab = np.loadtxt(os.path.join(GOLD, "healpix_ring_nside1.txt"))
    z, phi = gen.pix2zphi_ring(1)
    np.testing.assert_allclose(z, tab[:, 1] / 3.0, atol=1e-15)
    np.testing.assert_allclose(phi / np.pi, tab[:, 2], atol=1e-15)


def test_healpix_invariants():
    for ns in (1, 2, 4, 8, 16, 64):
        z, phi = gen.pix2zphi_ring(ns)
        v = gen.pix2vec_ring(ns)
        assert v.shape == (12 * ns * ns, 3)
        np.testing.assert_allclose(np.linalg.norm(v, axis=1), 1.0, atol=1e-14)
        assert np.abs(v.sum(0)).max() < 1e-11                      # centres balance
        assert len(np.unique(np.round(z, 12))) == 4 * ns - 1       # number of rings
        np.testing.assert_allclose(z, -z[::-1], atol=1e-15)        # north-south mirror
        assert np.all(np.diff(z) <= 1e-15)                         # RING: z non-increasing with p
        assert phi.min() >= 0 and phi.max() < 2 * np.pi
        # pixels per ring: 4i in caps, 4N in the belt
        _, counts = np.unique(np.round(z, 12), return_counts=True)
        counts = counts[::-1]
        exp = [4 * i for i in range(1, ns)] + [4 * ns] * (2 * ns + 1) + [4 * i for i in range(ns - 1, 0, -1)]
        assert counts.tolist() == exp
        # every ring is equally spaced in phi
        start = 0
        for c in exp:
            ph = phi[start:start + c]
            np.testing.assert_allclose(np.diff(ph), 2 * np.pi / c, atol=1e-12)
            start += c


def test_noise_sigma_R6():
    s = gen.noise_sigma(64)
    pix = np.sqrt(4 * np.pi / 49152) * 180 * 60 / np.pi
    assert abs(pix - 54.9678) < 1e-3
    np.testing.assert_allclose(s * pix, gen.DEPTHS_UK_ARCMIN)
    assert abs(s[9] - 0.1110) < 1e-4 and abs(s[0] - 0.6804) < 1e-4
    n = gen.ninv_f32(64)
    assert n.dtype == np.float32
    np.testing.assert_allclose(n, 1 / s ** 2, rtol=1e-7)


def test_latitude_regions_R17():
    reg = gen.latitude_regions(gen.pix2vec_ring(64))
    assert np.bincount(reg).tolist() == [17664, 14848, 16640]


def test_kmeans_rules():
    v = gen.pix2vec_ring(8)
    lab = gen.spherical_kmeans(v, 7, gen.rng_for("kmeans", 5))
    assert lab.dtype == np.int32 and lab.min() >= 0 and lab.max() < 7
    lab2 = gen.spherical_kmeans(v, 7, gen.rng_for("kmeans", 5))
    assert np.array_equal(lab, lab2)                               # seeded
    assert np.array_equal(gen.spherical_kmeans(v, 5000, gen.rng_for("kmeans", 1)), np.arange(768))   # K > npix
    assert np.all(gen.spherical_kmeans(v, 1, gen.rng_for("kmeans", 1)) == 0)
    sizes = np.bincount(lab, minlength=7)
    assert sizes.sum() == 768 and (sizes > 0).sum() >= 5
    # (that each pixel sits with its nearest centroid: tests/test_kmeans_oracle.py::test_generator_kmeans_rules, which has
    # the centroids of the last assignment from the K-means reference)


def test_workloads_shapes():
    w = gen.make_config(0)
    assert (w.npix, w.batch, w.ndata, w.maps.shape) == (768, 1, 1, (3, 768))
    assert w.Kmap.tolist() == [4, 2, 3]
    d = w.data()
    assert d.shape == (1, 15, 2, 768) and d.dtype == np.float32
    off = w.param_offsets()
    assert off.tolist() == [0, 9]
    g = gen.c3_grid()
    assert g.shape == (1024, 3) and len({tuple(r) for r in g}) == 1024
    assert sorted(set(g[:, 0])) == [10, 14, 18, 25, 34, 46, 63, 86, 117, 158, 215, 293, 398, 541, 736, 1000]
    w4 = gen.make_config(3, nside=16, ndata=3, batch=12)
    assert w4.nregion == 3 and w4.batch == 12 and w4.region_idx.dtype == np.uint8
    for m, k in zip(w4.maps, w4.Kmap):
        assert m.min() >= 0 and m.max() < k


def test_forward_model_is_unit_normalised():
    a_d, a_s = gen.mixing_columns([353.0, 23.0], 1.6, 19.0, -3.1)
    assert abs(a_d[0] - 1.0) < 1e-14 and abs(a_s[1] - 1.0) < 1e-14


def test_nested_superpixels_are_equal_area_compact_patches():
    """zphi2pix_nest (Gorski et al. 2005, restated): at a coarse nside the NESTED index partitions the pixel centres
    of a fine map into 12 nside_patch^2 patches of exactly (nside / nside_patch)^2 pixels each -- true only if faces,
    (ix, iy) and the bit interleave are all right -- and every patch is compact (its pixels lie within ~1.5 patch
    diagonals of their mean direction)."""
    for nside, npatch in ((8, 1), (16, 2), (32, 4), (64, 16), (64, 64)):
        m = gen.superpixel_map_ring(nside, npatch)
        counts = np.bincount(m, minlength=12 * npatch * npatch)
        assert counts.shape[0] == 12 * npatch * npatch and np.all(counts == (nside // npatch) ** 2)
    nside, npatch = 32, 4
    m = gen.superpixel_map_ring(nside, npatch)
    v = gen.pix2vec_ring(nside)
    size = np.sqrt(4 * np.pi / (12 * npatch * npatch))           # angular size of a patch
    for k in (0, 17, 100, 191):
        vk = v[m == k]
        c = vk.mean(axis=0)
        c /= np.linalg.norm(c)
        assert np.arccos(np.clip(vk @ c, -1, 1)).max() < 1.5 * size
    # at the map's own resolution the NESTED index is a permutation of the RING index with the known fixed points
    # of nside 1: pixel p of RING order is pixel p of NESTED order
    assert np.array_equal(gen.superpixel_map_ring(1, 1), np.arange(12))


def test_irregular_mask_and_multires_workload():
    w = gen.make_config(1, nside=16, multires=(8, 2, 4), holes=3)
    assert w.K_of_cfg(0) == [768, 48, 192]
    masked = (w.maps < 0).any(axis=0)
    assert np.array_equal(masked, (w.maps < 0).all(axis=0))         # a hole masks all three maps
    frac = masked.mean()
    assert 0.1 < frac < 0.5
    # no structure in RING order: masked runs of many different lengths, including single pixels
    edges = np.flatnonzero(np.diff(masked.astype(np.int8)))
    runs = np.diff(edges)
    assert len(np.unique(runs)) > 8 and runs.min() == 1
    # same seed, same mask; another seed, another mask
    assert np.array_equal(masked, (gen.make_config(1, nside=16, multires=(8, 2, 4), holes=3).maps < 0).any(axis=0))
    assert not np.array_equal(masked, (gen.make_config(1, nside=16, multires=(8, 2, 4), holes=4).maps < 0).any(axis=0))
