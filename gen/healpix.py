"""HEALPix RING pixel centres, restated from the published scheme (Gorski et al. 2005, cited PAPER.md:L29, L219).

No healpy in this image, so the RING formulas are written out.  Rings are counted from
the north pole, i = 1 .. 4N-1; ring i of a polar cap holds 4i pixels, every belt ring holds 4N.
"""
import numpy as np


def nside2npix(nside: int) -> int:
    return 12 * nside * nside


def _cap_ring(p: np.ndarray) -> np.ndarray:
    """Ring index i >= 1 of cap pixel p (counted from the pole): 2i(i-1) <= p < 2i(i+1)."""
    i = np.floor((1.0 + np.sqrt(1.0 + 2.0 * p.astype(np.float64))) / 2.0).astype(np.int64)
    # integer fix-up so that float rounding never misplaces a pixel
    i = np.where(2 * i * (i - 1) > p, i - 1, i)
    i = np.where(2 * i * (i + 1) <= p, i + 1, i)
    return i


def pix2zphi_ring(nside: int):
    """Return (z, phi) of every RING pixel centre, z = cos(colatitude), phi in [0, 2pi)."""
    n = int(nside)
    npix = nside2npix(n)
    ncap = 2 * n * (n - 1)
    p = np.arange(npix, dtype=np.int64)
    z = np.empty(npix, dtype=np.float64)
    phi = np.empty(npix, dtype=np.float64)

    north = p < ncap
    if north.any():
        pn = p[north]
        i = _cap_ring(pn)
        j = pn + 1 - 2 * i * (i - 1)                  # 1 .. 4i
        z[north] = 1.0 - (i * i) / (3.0 * n * n)
        phi[north] = (j - 0.5) * np.pi / (2.0 * i)

    belt = (p >= ncap) & (p < npix - ncap)
    pb = p[belt] - ncap
    i = pb // (4 * n) + n                             # n .. 3n
    j = pb % (4 * n) + 1                              # 1 .. 4n
    fodd = np.where(((i + n) % 2) == 1, 1.0, 0.5)
    z[belt] = (2 * n - i) * 2.0 / (3.0 * n)
    phi[belt] = (j - fodd) * np.pi / (2.0 * n)

    south = p >= npix - ncap
    if south.any():
        ps = npix - 1 - p[south]                      # mirror: counted from the south pole
        i = _cap_ring(ps)
        jm = ps + 1 - 2 * i * (i - 1)                 # 1 .. 4i counted backwards in phi
        j = 4 * i + 1 - jm
        z[south] = -1.0 + (i * i) / (3.0 * n * n)
        phi[south] = (j - 0.5) * np.pi / (2.0 * i)
    return z, phi


def pix2vec_ring(nside: int) -> np.ndarray:
    """Unit vectors [npix, 3] of RING pixel centres, n = (cos d cos a, cos d sin a, sin d)."""
    z, phi = pix2zphi_ring(nside)
    st = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([st * np.cos(phi), st * np.sin(phi), z], axis=1)


def zphi2pix_nest(nside: int, z: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """NESTED pixel index at resolution `nside` of the directions (z, phi), restated from the published scheme
    (Gorski et al. 2005): the sphere is twelve base faces, each an nside x nside grid whose cell (ix, iy) has the index
    face * nside^2 + bit-interleave(ix, iy).  Used to build multi-resolution super-pixel patches (Table 3,
    L328-L334): the NESTED index at a coarse nside is a partition into compact equal-area patches."""
    n = int(nside)
    assert n >= 1 and (n & (n - 1)) == 0, "NESTED needs a power-of-two nside"
    z = np.asarray(z, dtype=np.float64)
    za = np.abs(z)
    tt = np.mod(np.asarray(phi, dtype=np.float64), 2.0 * np.pi) / (0.5 * np.pi)      # [0, 4)
    face = np.empty(z.shape, dtype=np.int64)
    ix = np.empty(z.shape, dtype=np.int64)
    iy = np.empty(z.shape, dtype=np.int64)
    eq = za <= 2.0 / 3.0
    # equatorial belt
    t1 = n * (0.5 + tt[eq])
    t2 = n * z[eq] * 0.75
    jp = np.floor(t1 - t2).astype(np.int64)         # ascending edge line
    jm = np.floor(t1 + t2).astype(np.int64)         # descending edge line
    ifp, ifm = jp // n, jm // n
    face[eq] = np.where(ifp == ifm, (ifp & 3) + 4, np.where(ifp < ifm, ifp & 3, (ifm & 3) + 8))
    ix[eq] = jm & (n - 1)
    iy[eq] = n - (jp & (n - 1)) - 1
    # polar caps
    po = ~eq
    ntt = np.minimum(3, np.floor(tt[po]).astype(np.int64))
    tp = tt[po] - ntt
    tmp = n * np.sqrt(3.0 * (1.0 - za[po]))
    jp = np.minimum(n - 1, np.floor(tp * tmp).astype(np.int64))
    jm = np.minimum(n - 1, np.floor((1.0 - tp) * tmp).astype(np.int64))
    north = z[po] >= 0
    face[po] = np.where(north, ntt, ntt + 8)
    ix[po] = np.where(north, n - jm - 1, jp)
    iy[po] = np.where(north, n - jp - 1, jm)
    # interleave the bits of ix (even positions) and iy (odd positions)
    idx = np.zeros(z.shape, dtype=np.int64)
    for b in range(max(1, n.bit_length() - 1)):
        idx |= ((ix >> b) & 1) << (2 * b)
        idx |= ((iy >> b) & 1) << (2 * b + 1)
    return face * n * n + idx


def superpixel_map_ring(nside: int, nside_patch: int) -> np.ndarray:
    """int32 [npix]: for every RING pixel of the nside map, the NESTED index of the nside_patch super-pixel that holds
    its centre (`multires_clusters` of the paper, L607: a fixed baseline tiling with K = 12 nside_patch^2 patches)."""
    z, phi = pix2zphi_ring(nside)
    return zphi2pix_nest(nside_patch, z, phi).astype(np.int32)
