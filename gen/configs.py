"""The five BASELINE.json workloads as seeded recipes; all inputs synthetic.

A Workload carries exactly the buffers the C ABI takes (and the oracle takes the same ones):
  maps[nmap, npix] int32 cluster ids (-1 = masked), Kmap[nmap], cfg_maps[ncfg, 3] (a configuration is a
  triple of maps: beta_d, T_d, beta_s), region_idx[npix] uint8, cfg_of[B], data_of[B], ninv[F] fp32 and
  d[ndata, F, 2, npix] fp32 (built on demand: it can be GBs).
"""
from dataclasses import dataclass, field
import numpy as np

from .healpix import pix2vec_ring, nside2npix
from .kmeans import spherical_kmeans
from . import sky


def latitude_regions(vecs: np.ndarray) -> np.ndarray:
    """Stand-in for the Planck GAL masks (R17): |b|>40 -> 0, 20<|b|<=40 -> 1, |b|<=20 -> 2."""
    b = np.degrees(np.arcsin(np.clip(vecs[:, 2], -1.0, 1.0)))
    reg = np.full(vecs.shape[0], 2, dtype=np.uint8)
    reg[np.abs(b) > 20.0] = 1
    reg[np.abs(b) > 40.0] = 0
    return reg


_MAP_CACHE = {}


def cluster_map(vecs: np.ndarray, param: int, K: int, region_idx=None, nregion: int = 1, iters: int = 10):
    """One cluster map for spectral parameter `param` (0,1,2) with K patches (per region when regions are
    given: independent K-means per region, ids concatenated region after region, K capped at the region's
    pixel count).  Returns (labels int32 [npix], K_total).  Seeded, hence cached per process."""
    key = (vecs.shape[0], float(vecs[vecs.shape[0] // 3, 0]), int(param), int(K), int(nregion),
           None if region_idx is None else hash(np.asarray(region_idx).tobytes()), int(iters))
    if key not in _MAP_CACHE:
        lab, kt = _cluster_map(vecs, param, K, region_idx, nregion, iters)
        lab.setflags(write=False)
        _MAP_CACHE[key] = (lab, kt)
    lab, kt = _MAP_CACHE[key]
    return lab.copy(), kt


def _cluster_map(vecs: np.ndarray, param: int, K: int, region_idx, nregion: int, iters: int):
    npix = vecs.shape[0]
    if region_idx is None or nregion == 1:
        g = sky.rng_for("kmeans", (param * 1_000_003 + K) * 16)
        lab = spherical_kmeans(vecs, K, g, iters)
        return lab.astype(np.int32), int(min(K, npix))
    lab = np.empty(npix, dtype=np.int32)
    off = 0
    for r in range(nregion):
        sel = np.flatnonzero(region_idx == r)
        g = sky.rng_for("kmeans", (param * 1_000_003 + K) * 16 + r + 1)
        lr = spherical_kmeans(vecs[sel], K, g, iters, seed_from_pixels=True)
        lab[sel] = lr + off
        off += int(min(K, sel.size))
    return lab, off


def irregular_mask(vecs: np.ndarray, seed: int = 0, ndisc: int = 40, frac_pix: float = 0.03) -> np.ndarray:
    """bool [npix], True = masked: a Planck-like irregular mask made of a band of random width along the equator
    ("Galactic plane" with a ragged edge), `ndisc` point-source discs of random radius (0.5 .. 6 degrees) and isolated
    random pixels.  Stands in for the Planck GAL / point-source masks, which are not available
    here; its purpose is a mask with no structure in RING order."""
    g = sky.rng_for("mask", seed)
    npix = vecs.shape[0]
    lon = np.arctan2(vecs[:, 1], vecs[:, 0])
    edge = np.deg2rad(8.0 + 6.0 * np.sin(3.0 * lon + g.uniform(0, 2 * np.pi)) + 3.0 * np.sin(11.0 * lon + g.uniform(0, 2 * np.pi)))
    m = np.abs(np.arcsin(vecs[:, 2])) < edge
    centres = g.standard_normal((ndisc, 3))
    centres /= np.linalg.norm(centres, axis=1, keepdims=True)
    radii = np.deg2rad(g.uniform(0.5, 6.0, ndisc))
    for c, r in zip(centres, radii):
        m |= vecs @ c > np.cos(r)
    m |= g.random(npix) < frac_pix
    return m


def multires_maps(nside: int, nside_patch=(16, 4, 8)):
    """Multi-resolution super-pixel patches (Table 3): one NESTED super-pixel map per spectral
    parameter.  Returns (maps int32 [3, npix], K [3])."""
    from .healpix import superpixel_map_ring
    maps = np.stack([superpixel_map_ring(nside, min(int(n), nside)) for n in nside_patch])
    return np.ascontiguousarray(maps.astype(np.int32)), [12 * min(int(n), nside) ** 2 for n in nside_patch]


def c3_grid(seed: int = 3) -> np.ndarray:
    """The 16 x 8 x 8 = 1024 clustering grid of configs[2], in a seeded shuffled order; rows (K_bd, K_Td, K_bs)."""
    kbd = [int(round(10 ** (1 + 2 * i / 15))) for i in range(16)]
    kk = [1, 5, 10, 20, 50, 100, 200, 500]
    grid = np.array([(a, b, c) for a in kbd for b in kk for c in kk], dtype=np.int64)
    perm = sky.rng_for("shuffle", seed).permutation(len(grid))
    return grid[perm]


@dataclass
class Workload:
    name: str
    nside: int
    npix: int
    freqs: np.ndarray
    ninv: np.ndarray            # fp32 [F]
    sigma: np.ndarray           # fp64 [F]
    maps: np.ndarray            # int32 [nmap, npix]
    Kmap: np.ndarray            # int32 [nmap]
    cfg_maps: np.ndarray        # int32 [ncfg, 3]
    region_idx: np.ndarray      # uint8 [npix] or None
    nregion: int
    cfg_of: np.ndarray          # int32 [B]
    data_of: np.ndarray         # int32 [B]
    ndata: int
    truth: dict
    realizations: tuple = (0,)
    noiseless: bool = False
    _d: np.ndarray = field(default=None, repr=False)

    @property
    def batch(self) -> int:
        return int(self.cfg_of.shape[0])

    @property
    def nfreq(self) -> int:
        return int(self.freqs.shape[0])

    def K_of_cfg(self, c: int):
        return [int(self.Kmap[m]) for m in self.cfg_maps[c]]

    def param_offsets(self) -> np.ndarray:
        """int64 [B+1]: entry e owns params[off[e]:off[e+1]] = [beta_d x K0 ; T_d x K1 ; beta_s x K2]."""
        n = np.array([sum(self.K_of_cfg(int(c))) for c in self.cfg_of], dtype=np.int64)
        return np.concatenate([[0], np.cumsum(n)])

    def params_const(self, beta_d=1.54, T_d=20.0, beta_s=-3.0) -> np.ndarray:
        off = self.param_offsets()
        p = np.empty(off[-1], dtype=np.float64)
        for e, c in enumerate(self.cfg_of):
            K0, K1, K2 = self.K_of_cfg(int(c))
            o = off[e]
            p[o:o + K0] = beta_d
            p[o + K0:o + K0 + K1] = T_d
            p[o + K0 + K1:o + K0 + K1 + K2] = beta_s
        return p

    def params_jittered(self, seed: int = 0, scale: float = 1.0) -> np.ndarray:
        """Start values scattered around (1.54, 20, -3): exercises every cluster with a distinct value."""
        g = sky.rng_for("params", seed)
        p = self.params_const()
        off = self.param_offsets()
        for e, c in enumerate(self.cfg_of):
            K0, K1, K2 = self.K_of_cfg(int(c))
            o = off[e]
            p[o:o + K0] += scale * 0.05 * g.standard_normal(K0)
            p[o + K0:o + K0 + K1] += scale * 0.8 * g.standard_normal(K1)
            p[o + K0 + K1:o + K0 + K1 + K2] += scale * 0.05 * g.standard_normal(K2)
        return p

    def data(self) -> np.ndarray:
        if self._d is None:
            self._d = sky.synthesize(self.truth, self.freqs, None if self.noiseless else self.sigma,
                                     self.realizations)
        return self._d


def _base(nside: int):
    vecs = pix2vec_ring(nside)
    return vecs, nside2npix(nside), sky.BANDS_GHZ.copy(), sky.ninv_f32(nside), sky.noise_sigma(nside)


def make_config(idx: int, *, nside=None, batch=None, ndata=None, K=None, noiseless=False,
                cluster_truth=False, sky_seed: int = 1, multires=None, holes=None) -> Workload:
    """BASELINE.json configs[idx] (idx 0..4), optionally scaled down (nside / batch / ndata) for tests.

    0: tiny sky nside 8, K=(4,2,3).   1: nside 64, K=(500,50,100), one entry.
    2: nside 64 clustering scan, 1024 configurations from 32 distinct maps, one shared noise realisation.
    3: nside 64, 3 latitude regions, 64 configurations x 100 noise realisations.
    4: nside 128, K=(2000,200,400), 256 noise realisations (batch sweep {1,16,64,256} = prefixes).
    `cluster_truth=True` makes the truth constant per cluster of configuration 0.
    `multires=(n0, n1, n2)` (configs 0, 1, 4) replaces the K-means maps by NESTED super-pixel maps at those resolutions
    (Table 3); `holes=seed` masks an irregular, Planck-like set of pixels (-1 in all three maps)."""
    defaults = {0: (8, (4, 2, 3)), 1: (64, (500, 50, 100)), 2: (64, None), 3: (64, None), 4: (128, (2000, 200, 400))}
    nside = nside or defaults[idx][0]
    K = K or defaults[idx][1]
    vecs, npix, freqs, ninv, sigma = _base(nside)
    region_idx, nregion = None, 1
    if idx in (0, 1, 4):
        maps, Kmap = [], []
        if multires is not None:
            mm, Kmap = multires_maps(nside, multires)
            maps = [mm[0], mm[1], mm[2]]
        else:
            for prm in range(3):
                m, kt = cluster_map(vecs, prm, int(K[prm]))
                maps.append(m); Kmap.append(kt)
        cfg_maps = np.array([[0, 1, 2]], dtype=np.int32)
        nd = ndata or (256 if idx == 4 else 1)
        B = batch or nd
        cfg_of = np.zeros(B, dtype=np.int32)
        data_of = (np.arange(B) % nd).astype(np.int32)
        name = {0: "C1", 1: "C2", 4: "C5"}[idx]
    else:
        grid = c3_grid()
        if idx == 3:
            region_idx = latitude_regions(vecs); nregion = 3
            ncfg = 64
        else:
            ncfg = 1024
        if batch is not None and idx == 2:
            ncfg = min(ncfg, batch)
        grid = grid[:ncfg]
        maps, Kmap, key2map = [], [], {}
        cfg_maps = np.empty((ncfg, 3), dtype=np.int32)
        for c, kk in enumerate(grid):
            for prm in range(3):
                key = (prm, int(kk[prm]))
                if key not in key2map:
                    m, kt = cluster_map(vecs, prm, int(kk[prm]), region_idx, nregion)
                    key2map[key] = len(maps); maps.append(m); Kmap.append(kt)
                cfg_maps[c, prm] = key2map[key]
        if idx == 2:
            nd = ndata or 1
            cfg_of = np.arange(ncfg, dtype=np.int32)
            data_of = np.zeros(ncfg, dtype=np.int32)
            name = "C3"
        else:
            nd = ndata or 100
            # noise-major inside each configuration: entry = cfg * nd + realisation
            cfg_of = np.repeat(np.arange(ncfg, dtype=np.int32), nd)
            data_of = np.tile(np.arange(nd, dtype=np.int32), ncfg)
            if batch is not None:
                cfg_of, data_of = cfg_of[:batch], data_of[:batch]
            name = "C4"
    maps = np.ascontiguousarray(np.stack(maps).astype(np.int32))
    Kmap = np.array(Kmap, dtype=np.int32)
    if holes is not None:
        maps[:, irregular_mask(vecs, int(holes))] = -1
    if cluster_truth:
        tm = maps[cfg_maps[0]]
        truth = sky.draw_truth(npix, sky_seed, tm, [int(Kmap[m]) for m in cfg_maps[0]])
    else:
        truth = sky.draw_truth(npix, sky_seed)
    return Workload(name=name, nside=nside, npix=npix, freqs=freqs, ninv=ninv, sigma=sigma, maps=maps, Kmap=Kmap,
                    cfg_maps=cfg_maps, region_idx=region_idx, nregion=nregion, cfg_of=cfg_of, data_of=data_of,
                    ndata=int(nd), truth=truth, realizations=tuple(range(int(nd))), noiseless=noiseless)
