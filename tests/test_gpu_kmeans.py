"""f2: cs_spherical_kmeans (GPU, batched) against the K-means reference oracle/kmeans.py (pinned in
tests/test_kmeans_oracle.py) -- labels must agree bit for bit (index work).  The random numbers of the method (the
initial centroids) are drawn by gen's seeded generator and passed to both; that the generator's own maps equal the
reference's is a CPU test (tests/test_kmeans_oracle.py)."""
import numpy as np
import pytest

import gen
from gen import kmeans as gk
from gen import sky
from oracle import kmeans as ok

pytestmark = pytest.mark.gpu


def _gpu_cluster_maps(vecs, specs, region_idx=None, nregion=1, iters=10):
    """specs: list of (param, K).  Returns {spec: (labels int32 [npix], K_total)} computed like gen.cluster_map, with
    every K-means problem (one per region) of every spec in ONE batched GPU call."""
    import torch
    import paper_2604_08463_b200 as cs
    npix = vecs.shape[0]
    probs = []          # (spec index, region or -1, K, cent0 [K,3])
    trivial = {}        # (spec index, region) -> labels of the region's pixels when no K-means is needed
    for si, (param, K) in enumerate(specs):
        regs = [None] if (region_idx is None or nregion == 1) else list(range(nregion))
        for r in regs:
            sel = np.arange(npix) if r is None else np.flatnonzero(region_idx == r)
            seed = (param * 1_000_003 + K) * 16 + (0 if r is None else r + 1)
            g = sky.rng_for("kmeans", seed)
            if K >= sel.size:
                trivial[(si, r)] = np.arange(sel.size, dtype=np.int32)
            elif K == 1:
                trivial[(si, r)] = np.zeros(sel.size, dtype=np.int32)
            else:
                probs.append((si, -1 if r is None else r, K, gk.initial_centroids(vecs[sel], K, g, seed_from_pixels=r is not None)))
    labels = None
    if probs:
        Ks = np.array([p[2] for p in probs], dtype=np.int32)
        cent = torch.from_numpy(np.concatenate([p[3] for p in probs])).cuda()
        lab_d = torch.full((len(probs), npix), -7, dtype=torch.int32, device="cuda")
        reg_d = None if region_idx is None else torch.from_numpy(region_idx.astype(np.uint8)).cuda()
        cs.spherical_kmeans(torch.from_numpy(vecs).cuda(), Ks, cent, lab_d, iters=iters, region=reg_d,
                            prob_region=np.array([p[1] for p in probs], dtype=np.int32))
        torch.cuda.synchronize()
        labels = lab_d.cpu().numpy()
    out = {}
    for si, (param, K) in enumerate(specs):
        lab = np.empty(npix, dtype=np.int32)
        off = 0
        regs = [None] if (region_idx is None or nregion == 1) else list(range(nregion))
        for r in regs:
            sel = np.arange(npix) if r is None else np.flatnonzero(region_idx == r)
            if (si, r) in trivial:
                lr = trivial[(si, r)]
            else:
                j = next(i for i, p in enumerate(probs) if p[0] == si and p[1] == (-1 if r is None else r))
                lr = labels[j][sel]
                outside = np.ones(npix, dtype=bool)
                outside[sel] = False
                assert np.all(labels[j][outside] == -1)
            lab[sel] = lr + off
            off += int(min(K, sel.size))
        out[(param, K)] = (lab, off)
    return out


def _oracle_map(vecs, param, K, region_idx=None, nregion=1):
    def cent0(r, sel):
        seed = (param * 1_000_003 + K) * 16 + (0 if r is None else r + 1)
        return gk.initial_centroids(vecs[sel], K, sky.rng_for("kmeans", seed), seed_from_pixels=r is not None)
    return ok.patch_map(vecs, K, cent0, region_idx, nregion)


def _check(vecs, specs, region_idx=None, nregion=1):
    got = _gpu_cluster_maps(vecs, specs, region_idx, nregion)
    for param, K in specs:
        want, ktot = _oracle_map(vecs, param, K, region_idx, nregion)
        lab, k2 = got[(param, K)]
        assert k2 == ktot
        assert np.array_equal(lab, want), (param, K, int((lab != want).sum()))


def test_kmeans_labels_c1_c2():
    _check(gen.pix2vec_ring(8), [(0, 4), (1, 2), (2, 3)])
    _check(gen.pix2vec_ring(64), [(0, 500), (1, 50), (2, 100)])


def test_kmeans_labels_c3_grid_maps():
    """All 32 distinct maps of the clustering scan (16 + 8 + 8 values of K, from 1 to 1000) in one batched call."""
    grid = gen.c3_grid()
    specs = sorted({(prm, int(k[prm])) for k in grid for prm in range(3)})
    assert len(specs) == 32
    _check(gen.pix2vec_ring(64), specs)


def test_kmeans_labels_c4_regions():
    """Three latitude regions with independent K-means per region (seeded from region pixels), K capped at the
    region's pixel count, ids concatenated region after region."""
    vecs = gen.pix2vec_ring(32)
    reg = gen.latitude_regions(vecs)
    grid = gen.c3_grid()[:64]
    specs = sorted({(prm, int(k[prm])) for k in grid for prm in range(3)})
    _check(vecs, specs, reg, 3)


def test_kmeans_is_deterministic_and_handles_empty_patches():
    import torch
    import paper_2604_08463_b200 as cs
    vecs = gen.pix2vec_ring(16)
    g = sky.rng_for("misc", 41)
    cent0 = gk.initial_centroids(vecs, 40, g)
    cent0[7] = -cent0[3]
    cent0[8] = cent0[3]                       # a duplicate centroid: ties go to the lower id, patch 8 stays empty
    outs = []
    for _ in range(2):
        cent = torch.from_numpy(cent0.copy()).cuda()
        lab = torch.zeros((1, vecs.shape[0]), dtype=torch.int32, device="cuda")
        cs.spherical_kmeans(torch.from_numpy(vecs).cuda(), [40], cent, lab, iters=10)
        torch.cuda.synchronize()
        outs.append((lab.cpu().numpy(), cent.cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    lab_ref, cent_ref = ok.lloyd(vecs, cent0, iters=10)       # labels and final centroids of the reference, bit for bit
    assert np.array_equal(outs[0][0][0], lab_ref) and np.array_equal(outs[0][1], cent_ref)
    assert np.allclose(np.linalg.norm(outs[0][1], axis=1), 1.0, atol=1e-15)
    # no iteration: the duplicate loses every tie; one iteration: it was empty during the update and keeps its centroid
    res = {}
    for iters in (0, 1):
        cent = torch.from_numpy(cent0.copy()).cuda()
        lab = torch.zeros((1, vecs.shape[0]), dtype=torch.int32, device="cuda")
        cs.spherical_kmeans(torch.from_numpy(vecs).cuda(), [40], cent, lab, iters=iters)
        torch.cuda.synchronize()
        res[iters] = (lab.cpu().numpy(), cent.cpu().numpy())
    assert not np.any(res[0][0] == 8) and np.any(res[0][0] == 3) and np.array_equal(res[0][1], cent0)
    assert np.array_equal(res[1][1][8], cent0[8]) and not np.array_equal(res[1][1][3], cent0[3])


def test_kmeans_takes_more_than_65535_problems():
    """Problems beyond the 65535 of grid.y go in slices: here all the same problem, so every row of labels and every
    block of centroids equals the reference's."""
    import torch
    import paper_2604_08463_b200 as cs
    vecs = gen.pix2vec_ring(4)
    nprob, K = 65535 + 9, 3
    c0 = gk.initial_centroids(vecs, K, sky.rng_for("misc", 77))
    cent = torch.from_numpy(np.tile(c0, (nprob, 1))).cuda()
    lab = torch.full((nprob, vecs.shape[0]), -7, dtype=torch.int32, device="cuda")
    cs.spherical_kmeans(torch.from_numpy(vecs).cuda(), np.full(nprob, K, dtype=np.int32), cent, lab, iters=3)
    torch.cuda.synchronize()
    lab_ref, cent_ref = ok.lloyd(vecs, c0, iters=3)
    assert torch.equal(lab, torch.from_numpy(lab_ref).cuda().expand(nprob, -1))
    assert np.array_equal(cent.cpu().numpy().reshape(nprob, K, 3), np.broadcast_to(cent_ref, (nprob, K, 3)))
