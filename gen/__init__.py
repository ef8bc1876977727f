"""Seeded synthetic-input generators (LiteBIRD-shaped skies, HEALPix RING geometry, spherical K-means).

This package only *produces inputs*: pixel geometry, cluster maps, random sky fields, noise and the
forward data model d = A(beta) s + n (Eq. 1-2) needed to synthesise them.  It holds none
of the hot path's arithmetic (no likelihood, no GLS solve, no gradient, no cluster reduction), and neither
`oracle/` nor the CUDA library imports it: tests and `bench.py` call it and hand the same buffers to both.

Recipe and citations: DESIGN.md "Input recipe"; BASELINE.json `configs`; SURVEY.md 8(d).
"""
from .healpix import nside2npix, pix2vec_ring, pix2zphi_ring, zphi2pix_nest, superpixel_map_ring  # noqa: F401
from .kmeans import spherical_kmeans  # noqa: F401
from .sky import (  # noqa: F401
    BANDS_GHZ, DEPTHS_UK_ARCMIN, NU0_DUST_GHZ, NU0_SYNC_GHZ, T_CMB_K,
    noise_sigma, ninv_f32, draw_truth, mixing_columns, synthesize, noise_field, rng_for,
)
from .configs import (  # noqa: F401
    latitude_regions, cluster_map, c3_grid, make_config, Workload, irregular_mask, multires_maps,
)
