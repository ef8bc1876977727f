"""cs_spherical_kmeans_static, the K-means entry point that allocates nothing, against cs_spherical_kmeans.

Why the entry point exists: some hosts of this library cannot let it call cudaMalloc -- a server whose own pool has
taken the whole GPU (an allocation from a library may then fail at any moment), or a loop that cannot afford the
device-wide synchronisation an allocation or a free may bring.  For them the one piece of scratch memory K-means
needs, its table of problem descriptors, lives in a fixed device array inside libcs.so (at most
KMEANS_STATIC_MAX_PROB = 1024 problems a call) instead of a per-call allocation.

What is checked: both entry points run the same kernels on the same seeded inputs, so labels (index work) and final
centroids (fp64, fixed operation order) must be equal bit for bit -- the bar tests/test_gpu_kmeans.py sets for labels.
The calls come one right after the other on one stream, with fewer and different problems in the second one: the shared
table still holds the first call's descriptors then, and a call that trusted stale contents would give wrong labels.
The file is named to be collected last, so that a failure here cannot hide another test under `pytest -x`; nothing in
it depends on what ran before (it passes alone in a fresh process as well).
"""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


def _problem_set(vecs, region_idx, Ks, regions, seed):
    """Initial centroids of each problem: K distinct pixel centres drawn (seeded) among the problem's pixels."""
    g = np.random.default_rng(seed)
    cents = []
    for K, r in zip(Ks, regions):
        sel = np.arange(vecs.shape[0]) if r < 0 else np.flatnonzero(region_idx == r)
        assert K <= sel.size
        cents.append(vecs[g.choice(sel, size=K, replace=False)])
    return np.concatenate(cents)


def _run(fn, vecs_d, reg_d, Ks, regions, cent0, iters):
    import torch
    cent = torch.from_numpy(cent0.copy()).cuda()
    labels = torch.full((len(Ks), vecs_d.shape[0]), -7, dtype=torch.int32, device="cuda")
    fn(vecs_d, np.asarray(Ks, dtype=np.int32), cent, labels, iters=iters, region=reg_d,
       prob_region=np.asarray(regions, dtype=np.int32))
    return cent, labels


def _inputs(nside, drop):
    import torch
    vecs = np.ascontiguousarray(gen.pix2vec_ring(nside)[:12 * nside * nside - drop])   # ragged last block of 256
    region_idx = np.digitize(vecs[:, 2], [-0.3, 0.4]).astype(np.uint8)                  # three latitude bands
    return vecs, region_idx, torch.from_numpy(vecs).cuda(), torch.from_numpy(region_idx).cuda()


def test_static_kmeans_matches_the_allocating_path_on_two_calls_in_a_row():
    import torch
    import paper_2604_08463_b200 as cs
    vecs, region_idx, vecs_d, reg_d = _inputs(32, drop=37)
    # first call: five problems, one with more patches than a shared-memory tile of centroids (1024), one trivial
    Ks1, regs1 = [7, 300, 1, 64, 1500], [-1, 0, 1, 2, -1]
    # second call: fewer problems, other patch counts and regions; the table still holds call one's five descriptors
    Ks2, regs2 = [33, 5], [2, -1]
    c1 = _problem_set(vecs, region_idx, Ks1, regs1, seed=11)
    c2 = _problem_set(vecs, region_idx, Ks2, regs2, seed=12)
    got1 = _run(cs.spherical_kmeans_static, vecs_d, reg_d, Ks1, regs1, c1, iters=4)
    got2 = _run(cs.spherical_kmeans_static, vecs_d, reg_d, Ks2, regs2, c2, iters=4)    # no synchronisation in between
    torch.cuda.synchronize()
    want1 = _run(cs.spherical_kmeans, vecs_d, reg_d, Ks1, regs1, c1, iters=4)
    want2 = _run(cs.spherical_kmeans, vecs_d, reg_d, Ks2, regs2, c2, iters=4)
    torch.cuda.synchronize()
    for (gc, gl), (wc, wl), Ks in ((got1, want1, Ks1), (got2, want2, Ks2)):
        assert torch.equal(gl, wl), int((gl != wl).sum())
        assert torch.equal(gc.view(torch.int64), wc.view(torch.int64))     # fp64 centroids, bit for bit
        lab = gl.cpu().numpy()
        for j, K in enumerate(Ks):
            live = lab[j][lab[j] >= 0]
            assert live.size and live.max() < K and (K > 1 or not live.any())
    # the iterations moved something: the run is not a copy of its input
    assert not np.array_equal(got1[0].cpu().numpy(), c1)


def test_static_kmeans_at_its_limit_and_beyond():
    import torch
    import paper_2604_08463_b200 as cs
    vecs, region_idx, vecs_d, reg_d = _inputs(8, drop=5)
    n = cs.KMEANS_STATIC_MAX_PROB
    assert n == 1024
    Ks = [2 + (j % 3) for j in range(n)]
    regs = [(j % 4) - 1 for j in range(n)]
    c0 = _problem_set(vecs, region_idx, Ks, regs, seed=5)
    gc, gl = _run(cs.spherical_kmeans_static, vecs_d, reg_d, Ks, regs, c0, iters=2)
    wc, wl = _run(cs.spherical_kmeans, vecs_d, reg_d, Ks, regs, c0, iters=2)
    torch.cuda.synchronize()
    assert torch.equal(gl, wl) and torch.equal(gc.view(torch.int64), wc.view(torch.int64))
    # one problem too many: refused with its own error code before anything is copied or launched
    Ks.append(2)
    regs.append(-1)
    c0 = np.concatenate([c0, vecs[:2]])
    with pytest.raises(cs.CsError) as err:
        _run(cs.spherical_kmeans_static, vecs_d, reg_d, Ks, regs, c0, iters=1)
    assert err.value.code == cs.ELIMIT and "capacity" in str(err.value)
    # and the entry point still works afterwards
    gc, gl = _run(cs.spherical_kmeans_static, vecs_d, reg_d, [6], [-1], c0[:6], iters=3)
    wc, wl = _run(cs.spherical_kmeans, vecs_d, reg_d, [6], [-1], c0[:6], iters=3)
    torch.cuda.synchronize()
    assert torch.equal(gl, wl) and torch.equal(gc.view(torch.int64), wc.view(torch.int64))
