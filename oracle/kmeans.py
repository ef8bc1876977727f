"""ctypes loader for the CPU fp64 reference of spherical K-means patching (oracle/kmeans_oracle.c, f2).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs.  The product
package never imports this module, and this module imports neither the product nor the input generator: the initial
centroids (the method's random draw) are passed in.

PAPER.md:L93-L104 (patches = nearest centroid by angular distance, centroid = normalised mean, Lloyd iterations) and
L299 (more patches than pixels: every pixel its own patch); the readings the paper leaves open are DESIGN.md R15 and
are listed at the top of the C file.  Pinned in tests/test_kmeans_oracle.py.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kmeans_oracle.c")
_LIB = os.path.join(_HERE, "libkmeans_oracle.so")


def build(force: bool = False) -> str:
    """gcc, no fast-math, no contraction of a*b+c into a fused multiply-add (the dot product's roundings are part of
    the definition); OpenMP only splits the independent pixel loop of the assignment."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.orc_km_assign.restype = None
        L.orc_km_assign.argtypes = [i64, vp, i32, vp, vp]
        L.orc_km_update.restype = C.c_int
        L.orc_km_update.argtypes = [i64, vp, vp, i32, vp]
        L.orc_km_objective.restype = C.c_double
        L.orc_km_objective.argtypes = [i64, vp, vp, vp]
        L.orc_km_lloyd.restype = C.c_int
        L.orc_km_lloyd.argtypes = [i64, vp, i32, vp, i32, vp, vp]
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def assign(vecs, cent):
    """labels int32 [n]: the patch whose centroid has the largest dot product with the pixel, ties to the lowest id."""
    vecs, cent = _f64(vecs), _f64(cent)
    lab = np.empty(vecs.shape[0], dtype=np.int32)
    lib().orc_km_assign(vecs.shape[0], vecs.ctypes.data, cent.shape[0], cent.ctypes.data, lab.ctypes.data)
    return lab


def update(vecs, labels, cent):
    """New centroids [K,3]: normalised mean of each patch's pixels; a patch without pixels keeps its centroid."""
    vecs, out = _f64(vecs), _f64(cent).copy()
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    assert labels.min() >= 0 and labels.max() < out.shape[0]
    if lib().orc_km_update(vecs.shape[0], vecs.ctypes.data, labels.ctypes.data, out.shape[0], out.ctypes.data) != 0:
        raise MemoryError("orc_km_update")
    return out


def objective(vecs, labels, cent):
    """sum_p n_p . c_label(p)."""
    vecs, cent = _f64(vecs), _f64(cent)
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    return float(lib().orc_km_objective(vecs.shape[0], vecs.ctypes.data, labels.ctypes.data, cent.ctypes.data))


def lloyd(vecs, cent0, iters=10, want_objective=False):
    """One assignment with cent0, then `iters` Lloyd iterations.  Returns (labels [n], centroids [K,3]) and, when asked,
    the objective after each of the iters + 1 assignments."""
    vecs, cent = _f64(vecs), _f64(cent0).copy()
    lab = np.empty(vecs.shape[0], dtype=np.int32)
    obj = np.empty(iters + 1, dtype=np.float64) if want_objective else None
    rc = lib().orc_km_lloyd(vecs.shape[0], vecs.ctypes.data, cent.shape[0], cent.ctypes.data, int(iters), lab.ctypes.data,
                            None if obj is None else obj.ctypes.data)
    if rc != 0:
        raise MemoryError("orc_km_lloyd")
    return (lab, cent, obj) if want_objective else (lab, cent)


def patch_map(vecs, K, cent0_of_region, region_idx=None, nregion=1, iters=10):
    """Patch map of one spectral parameter: K patches on the whole pixel set, or, with regions, K patches on each region
    independently (regions are processed independently), patch ids running on from region to region.
    cent0_of_region(r, sel) returns the initial centroids [K,3] of the problem on pixels `sel` (r = None without
    regions); it is only called when a K-means problem is actually solved.  A problem with K >= its number of pixels
    gives every pixel its own patch (L299).  Returns (labels int32 [npix], total number of patches)."""
    vecs = _f64(vecs)
    npix = vecs.shape[0]
    regions = [None] if (region_idx is None or nregion == 1) else list(range(nregion))
    labels = np.empty(npix, dtype=np.int32)
    first = 0
    for r in regions:
        sel = np.arange(npix) if r is None else np.flatnonzero(np.asarray(region_idx) == r)
        if K >= sel.size:
            lab = np.arange(sel.size, dtype=np.int32)
        else:
            lab, _ = lloyd(vecs[sel], cent0_of_region(r, sel), iters)
        labels[sel] = lab + first
        first += int(min(K, sel.size))
    return labels, first
