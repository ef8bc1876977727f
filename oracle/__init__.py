"""ctypes loader for the CPU fp64 oracle (oracle/cs_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product package never imports this module.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cs_oracle.c")
_LIB = os.path.join(_HERE, "libcs_oracle.so")

UNITS_KCMB = 0
UNITS_LITERAL = 1


def build(force: bool = False) -> str:
    """Compile cs_oracle.c with gcc (no fast-math; OpenMP only parallelises the independent pixel loop)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _CModel(C.Structure):
    _fields_ = [("nfreq", C.c_int32), ("freqs_ghz", C.POINTER(C.c_double)), ("nu0_dust_ghz", C.c_double),
                ("nu0_sync_ghz", C.c_double), ("t_cmb_k", C.c_double), ("units", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dbl = C.c_double
        pm = C.POINTER(_CModel)
        L.orc_krj2kcmb.restype = dbl; L.orc_krj2kcmb.argtypes = [dbl, dbl]
        for nm, n in (("orc_sed_dust", 3), ("orc_sed_sync", 2), ("orc_dsed_dust_dbeta", 3),
                      ("orc_dsed_dust_dT", 3), ("orc_dsed_sync_dbeta", 2)):
            f = getattr(L, nm); f.restype = dbl; f.argtypes = [pm] + [dbl] * n
        L.orc_mixing_matrix.restype = None
        L.orc_mixing_matrix.argtypes = [pm, dbl, dbl, dbl, C.c_void_p, C.c_void_p]
        L.orc_pixel.restype = C.c_int
        L.orc_pixel.argtypes = [pm, C.c_void_p, C.c_void_p, C.c_void_p, dbl, dbl, dbl] + [C.c_void_p] * 4
        L.orc_nll_grad.restype = C.c_int
        L.orc_nll_grad.argtypes = [pm, C.c_int64] + [C.c_void_p] * 8 + [C.c_int32] + [C.c_void_p] * 5
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


class Model:
    """Frequencies [GHz], reference frequencies, T_cmb and unit convention (R2, R3)."""

    def __init__(self, freqs_ghz, nu0_dust=353.0, nu0_sync=23.0, t_cmb=2.7255, units=UNITS_KCMB):
        self.freqs = np.ascontiguousarray(freqs_ghz, dtype=np.float64)
        self.c = _CModel(len(self.freqs), self.freqs.ctypes.data_as(C.POINTER(C.c_double)),
                         float(nu0_dust), float(nu0_sync), float(t_cmb), int(units))
        self.nfreq = len(self.freqs)

    @property
    def ref(self):
        return C.byref(self.c)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def krj2kcmb(nu_ghz, t_cmb=2.7255):
    return lib().orc_krj2kcmb(float(nu_ghz), float(t_cmb))


def sed_dust(m, nu, beta_d, T_d):
    return lib().orc_sed_dust(m.ref, float(nu), float(beta_d), float(T_d))


def sed_sync(m, nu, beta_s):
    return lib().orc_sed_sync(m.ref, float(nu), float(beta_s))


def dsed_dust_dbeta(m, nu, beta_d, T_d):
    return lib().orc_dsed_dust_dbeta(m.ref, float(nu), float(beta_d), float(T_d))


def dsed_dust_dT(m, nu, beta_d, T_d):
    return lib().orc_dsed_dust_dT(m.ref, float(nu), float(beta_d), float(T_d))


def dsed_sync_dbeta(m, nu, beta_s):
    return lib().orc_dsed_sync_dbeta(m.ref, float(nu), float(beta_s))


def mixing_matrix(m, beta_d, T_d, beta_s):
    """A [F,3] and dA [3,F] (d a_d/d beta_d, d a_d/d T_d, d a_s/d beta_s)."""
    A = np.empty((m.nfreq, 3)); dA = np.empty((3, m.nfreq))
    lib().orc_mixing_matrix(m.ref, float(beta_d), float(T_d), float(beta_s), _p(A), _p(dA))
    return A, dA


def pixel(m, ninv, dq, du, beta_d, T_d, beta_s):
    """One pixel: returns dict(s[3,2], ll, g[3], gs[3], rc)."""
    ninv = np.ascontiguousarray(ninv, dtype=np.float64)
    dq = np.ascontiguousarray(dq, dtype=np.float64); du = np.ascontiguousarray(du, dtype=np.float64)
    s = np.empty((3, 2)); ll = np.empty(1); g = np.empty(3); gs = np.empty(3)
    rc = lib().orc_pixel(m.ref, _p(ninv), _p(dq), _p(du), float(beta_d), float(T_d), float(beta_s),
                         _p(s), _p(ll), _p(g), _p(gs))
    return {"s": s, "ll": float(ll[0]), "g": g, "gs": gs, "rc": rc}


def nll_grad(m, d, ninv, idx, K, params, region=None, nregion=1, want_grad=True, want_maps=False, want_tol=False):
    """One batch entry.  d float32 [F,2,npix]; ninv float32 [F]; idx int32 [3,npix]; K [3]; params float64 [Ktot].
    Returns dict(rc, nll[nregion], grad, maps[3,2,npix], absg, gscale)."""
    d = np.ascontiguousarray(d, dtype=np.float32)
    F, two, npix = d.shape
    assert F == m.nfreq and two == 2
    ninv = np.ascontiguousarray(ninv, dtype=np.float32)
    idx = [np.ascontiguousarray(idx[i], dtype=np.int32) for i in range(3)]
    K = np.ascontiguousarray(K, dtype=np.int32)
    params = np.ascontiguousarray(params, dtype=np.float64)
    Ktot = int(K.sum())
    assert params.shape[0] == Ktot
    if region is not None:
        region = np.ascontiguousarray(region, dtype=np.uint8)
    nll = np.empty(nregion)
    grad = np.empty(Ktot) if want_grad else None
    maps = np.empty((3, 2, npix)) if want_maps else None
    absg = np.empty(Ktot) if want_tol else None
    gscale = np.empty(Ktot) if want_tol else None
    rc = lib().orc_nll_grad(m.ref, npix, _p(d), _p(ninv), _p(idx[0]), _p(idx[1]), _p(idx[2]), _p(K), _p(params),
                            _p(region), int(nregion), _p(nll), _p(grad), _p(maps), _p(absg), _p(gscale))
    return {"rc": rc, "nll": nll, "grad": grad, "maps": maps, "absg": absg, "gscale": gscale}


def num_threads() -> int:
    return lib().orc_num_threads()


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))
