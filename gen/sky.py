"""Synthetic LiteBIRD-shaped polarised skies: truth fields, forward data model, white noise.

Stands in for the paper's PySM3 / LiteBIRD simulations, which are not in this
container.  Distributions follow BASELINE.json `configs[0]`; noise conversion follows SURVEY.md 8(c) R6.
The forward model below (Eq. 1-2 with the R1 correction and the K_RJ->K_CMB factor of R2) is used ONLY to
synthesise `d`; it is written independently of both `oracle/` and the CUDA tables.
"""
import numpy as np

BANDS_GHZ = np.array([40., 50., 60., 68., 78., 89., 100., 119., 140., 166., 195., 235., 280., 337., 402.])
DEPTHS_UK_ARCMIN = np.array([37.4, 33.5, 21.3, 19.9, 15.6, 12.3, 10.5, 8.4, 6.4, 6.1, 7.6, 10.7, 18.8, 31.3, 44.5])
NU0_DUST_GHZ = 353.0
NU0_SYNC_GHZ = 23.0
T_CMB_K = 2.7255
_H_OVER_K = 6.62607015e-34 / 1.380649e-23 * 1e9      # K per GHz

_PURPOSE = {"sky": 1, "noise": 2, "kmeans": 3, "shuffle": 4, "params": 5, "misc": 6, "mask": 7}


def rng_for(purpose: str, index: int = 0) -> np.random.Generator:
    """Counter-based stream keyed by (purpose, index): Philox-4x64."""
    return np.random.Generator(np.random.Philox(key=[_PURPOSE[purpose], int(index) & (2**64 - 1)]))


def noise_sigma(nside: int, depths=DEPTHS_UK_ARCMIN) -> np.ndarray:
    """Per-pixel white-noise sigma [uK] per band: depth / sqrt(pixel area in arcmin^2) (R6)."""
    npix = 12 * nside * nside
    pix_arcmin = np.sqrt(4.0 * np.pi / npix) * (180.0 * 60.0 / np.pi)
    return np.asarray(depths, dtype=np.float64) / pix_arcmin


def ninv_f32(nside: int, depths=DEPTHS_UK_ARCMIN) -> np.ndarray:
    """N^-1 diagonal per band, fp32 as the library and the oracle both receive it."""
    s = noise_sigma(nside, depths)
    return (1.0 / (s * s)).astype(np.float32)


def _krj2kcmb(nu_ghz):
    x = _H_OVER_K * np.asarray(nu_ghz, dtype=np.float64) / T_CMB_K
    return np.expm1(x) ** 2 / (x * x * np.exp(x))


def mixing_columns(freqs_ghz, beta_d, T_d, beta_s, kcmb: bool = True):
    """Dust and synchrotron columns of A for arrays of parameters: returns (a_d, a_s), shape [F, ...]."""
    nu = np.asarray(freqs_ghz, dtype=np.float64).reshape((-1,) + (1,) * np.ndim(beta_d))
    beta_d = np.asarray(beta_d, dtype=np.float64)[None]
    T_d = np.asarray(T_d, dtype=np.float64)[None]
    beta_s = np.asarray(beta_s, dtype=np.float64)[None]
    planck = np.expm1(_H_OVER_K * NU0_DUST_GHZ / T_d) / np.expm1(_H_OVER_K * nu / T_d)
    a_d = (nu / NU0_DUST_GHZ) ** (beta_d + 1.0) * planck
    a_s = (nu / NU0_SYNC_GHZ) ** beta_s
    if kcmb:
        a_d = a_d * (_krj2kcmb(nu) / _krj2kcmb(NU0_DUST_GHZ))
        a_s = a_s * (_krj2kcmb(nu) / _krj2kcmb(NU0_SYNC_GHZ))
    return a_d, a_s


def draw_truth(npix: int, seed: int = 1, cluster_maps=None, K=None):
    """Random truth fields.  Per pixel by default; with `cluster_maps` ([3,npix] int32, K=[K0,K1,K2]) the
    spectral parameters are constant per cluster (the 'known by construction' sky of PAPER.md:L287).
    Returns dict with beta_d, T_d, beta_s [npix] and s [3, 2, npix] (cmb, dust@nu0d, sync@nu0s; Q,U) in uK."""
    g = rng_for("sky", seed)
    if cluster_maps is None:
        beta_d = 1.54 + 0.1 * g.standard_normal(npix)
        T_d = 20.0 + 1.0 * g.standard_normal(npix)
        beta_s = -3.0 + 0.1 * g.standard_normal(npix)
        per_cluster = None
    else:
        cm = np.asarray(cluster_maps)
        pc = [1.54 + 0.1 * g.standard_normal(K[0]), 20.0 + 1.0 * g.standard_normal(K[1]),
              -3.0 + 0.1 * g.standard_normal(K[2])]
        beta_d, T_d, beta_s = (pc[i][np.maximum(cm[i], 0)] for i in range(3))
        per_cluster = pc
    s = np.empty((3, 2, npix))
    s[0] = 0.5 * g.standard_normal((2, npix))
    for c, med in ((1, 10.0), (2, 5.0)):
        amp = med * np.exp(g.standard_normal(npix))
        psi = 2.0 * np.pi * g.random(npix)
        s[c, 0] = amp * np.cos(psi)
        s[c, 1] = amp * np.sin(psi)
    return {"beta_d": beta_d, "T_d": T_d, "beta_s": beta_s, "s": s, "per_cluster": per_cluster}


def noise_field(nfreq: int, npix: int, realization: int) -> np.ndarray:
    """Unit-variance white noise [F, 2, npix] for realisation r (stream 'noise', index r)."""
    return rng_for("noise", realization).standard_normal((nfreq, 2, npix))


def synthesize(truth, freqs_ghz=BANDS_GHZ, sigma=None, realizations=(0,), kcmb: bool = True) -> np.ndarray:
    """d[ndata, F, 2, npix] fp32 = A(beta_p) s_p + sigma_f * n  (Eq. 1).  `sigma=None` -> noiseless."""
    a_d, a_s = mixing_columns(freqs_ghz, truth["beta_d"], truth["T_d"], truth["beta_s"], kcmb)   # [F, npix]
    s = truth["s"]
    sig = s[0][None] + a_d[:, None, :] * s[1][None] + a_s[:, None, :] * s[2][None]               # [F, 2, npix]
    F, _, npix = sig.shape
    out = np.empty((len(realizations), F, 2, npix), dtype=np.float32)
    for i, r in enumerate(realizations):
        if sigma is None:
            out[i] = sig
        else:
            out[i] = sig + np.asarray(sigma)[:, None, None] * noise_field(F, npix, r)
    return out
