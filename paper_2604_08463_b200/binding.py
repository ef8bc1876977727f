"""Thin ctypes binding of libcs (include/cs.h): argument marshalling only, same names as the C ABI.

PyTorch supplies device memory and streams; every step of the hot path runs in the CUDA kernels of
csrc/.  There is no CPU fallback: loading fails loudly when libcs.so is missing and cannot be built.
"""
import ctypes as C
import os
import numpy as np

from . import build as _build

OK, EINVAL, EINDEX, EDOMAIN, ESINGULAR, ECUDA, ENOMEM, ELIMIT = 0, -1, -2, -3, -4, -5, -6, -7
KMEANS_STATIC_MAX_PROB = 1024
UNITS_KCMB, UNITS_LITERAL = 0, 1
OPT_LAYOUT, OPT_FORM, OPT_MIN_FILL, OPT_COPY_LIMIT_MB, OPT_PIXEL_BETA = 1, 2, 3, 4, 5
PIXBETA_AUTO, PIXBETA_OFF = 0, 1
LAYOUT_AUTO, LAYOUT_INPLACE, LAYOUT_SORTED = 0, 1, 2
FORM_AUTO, FORM_DIRECT = 0, 1
METHOD_ADATOPK, METHOD_LBFGS = 0, 1

EXPORTS = ["cs_create", "cs_destroy", "cs_set_option", "cs_layout_info", "cs_model_constants", "cs_set_clusters", "cs_set_data", "cs_set_batch", "cs_param_offsets",
           "cs_build_sed_tables", "cs_spectral_like_grad", "cs_spectral_misfit", "cs_cell_moments", "cs_spectral_like_grad_cells", "cs_component_maps", "cs_cmb_residual_maps", "cs_cmb_variance", "cs_optimize",
           "cs_opt_defaults", "cs_eval_host", "cs_spherical_kmeans", "cs_spherical_kmeans_static", "cs_check", "cs_profile", "cs_profile_read", "cs_strerror", "cs_workspace_bytes", "cs_kernel_launches",
           "cs_version"]


class CsModel(C.Structure):
    _fields_ = [("nfreq", C.c_int32), ("freqs_ghz", C.POINTER(C.c_double)), ("nu0_dust_ghz", C.c_double),
                ("nu0_sync_ghz", C.c_double), ("t_cmb_k", C.c_double), ("units", C.c_int32), ("npix", C.c_int64)]


class CsOpt(C.Structure):
    _fields_ = [("iters", C.c_int32), ("ls_max", C.c_int32), ("lr", C.c_double), ("beta1", C.c_double),
                ("beta2", C.c_double), ("eps", C.c_double), ("ls_c1", C.c_double), ("safe_lo", C.c_double),
                ("safe_hi", C.c_double), ("ls_noise", C.c_double), ("topk", C.c_double), ("method", C.c_int32),
                ("history", C.c_int32)]


class CsError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} ({code})")


_lib = None


def lib():
    """Loads (building first if stale and nvcc is present) libcs.so; raises if it cannot."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.stale():
        try:
            path = _build.build()
        except Exception as exc:  # no nvcc on the box: use the shipped .so if there is one
            if not os.path.exists(path):
                raise RuntimeError(f"libcs.so is missing and could not be built: {exc}") from exc
    L = C.CDLL(path)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    sig = {
        "cs_create": (C.c_int, [C.POINTER(vp), C.POINTER(CsModel)]),
        "cs_destroy": (C.c_int, [vp]),
        "cs_set_option": (C.c_int, [vp, i32, C.c_double]),
        "cs_layout_info": (C.c_int, [vp, i32, C.POINTER(i32), C.POINTER(i32), C.POINTER(C.c_double)]),
        "cs_model_constants": (C.c_int, [vp, vp, vp, vp, vp, C.POINTER(C.c_double)]),
        "cs_set_clusters": (C.c_int, [vp, i32, vp, vp, i32, vp, vp, i32]),
        "cs_set_data": (C.c_int, [vp, i32, vp, vp]),
        "cs_set_batch": (C.c_int, [vp, i32, vp, vp]),
        "cs_param_offsets": (C.c_int, [vp, vp]),
        "cs_build_sed_tables": (C.c_int, [vp, vp, vp]),
        "cs_spectral_like_grad": (C.c_int, [vp, vp, vp, vp]),
        "cs_spectral_misfit": (C.c_int, [vp, vp, vp]),
        "cs_cell_moments": (C.c_int, [vp, vp]),
        "cs_spectral_like_grad_cells": (C.c_int, [vp, vp, vp, vp]),
        "cs_component_maps": (C.c_int, [vp, i32, vp, vp, vp]),
        "cs_cmb_residual_maps": (C.c_int, [vp, i32, vp, vp, vp, vp]),
        "cs_cmb_variance": (C.c_int, [vp, vp, vp]),
        "cs_optimize": (C.c_int, [vp, vp, vp, vp, C.POINTER(CsOpt), vp, vp]),
        "cs_opt_defaults": (None, [C.POINTER(CsOpt)]),
        "cs_eval_host": (C.c_int, [vp, i32, vp, vp, vp, vp, vp]),
        "cs_spherical_kmeans": (C.c_int, [i64, vp, vp, i32, vp, vp, vp, i32, vp, vp]),
        "cs_spherical_kmeans_static": (C.c_int, [i64, vp, vp, i32, vp, vp, vp, i32, vp, vp]),
        "cs_check": (C.c_int, [vp, vp]),
        "cs_profile": (C.c_int, [vp, C.c_int]),
        "cs_profile_read": (C.c_int, [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64)]),
        "cs_strerror": (C.c_char_p, [C.c_int]),
        "cs_workspace_bytes": (i64, [vp]),
        "cs_kernel_launches": (i64, [vp]),
        "cs_version": (C.c_int, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


def strerror(code: int) -> str:
    return lib().cs_strerror(int(code)).decode()


def _chk(code, where):
    if code != OK:
        raise CsError(code, where)


def _hp(a):
    """Host pointer of a contiguous numpy array (or None)."""
    return None if a is None else a.ctypes.data_as(C.c_void_p)


_NP_OF = {"float64": np.float64, "float32": np.float32, "int32": np.int32, "uint8": np.uint8}


def _ptr(t, dtype=None, device=None, numel=None, what="argument"):
    """Raw pointer of a torch tensor (device or host), a numpy array, an int, or None.  The C ABI takes untyped
    pointers: dtype ("float64", ...), device ("cuda" / "cpu") and the least element count are checked here."""
    if t is None:
        return None
    if isinstance(t, int):
        return C.c_void_p(t)
    if isinstance(t, np.ndarray):
        if not t.flags["C_CONTIGUOUS"]:
            raise ValueError(f"{what}: array must be C-contiguous")
        if dtype is not None and t.dtype != _NP_OF[dtype]:
            raise TypeError(f"{what}: expected {dtype}, got {t.dtype}")
        if device == "cuda":
            raise TypeError(f"{what}: expected a CUDA tensor, got a numpy array")
        if numel is not None and t.size < numel:
            raise ValueError(f"{what}: {t.size} elements, need {numel}")
        return t.ctypes.data_as(C.c_void_p)
    if not t.is_contiguous():
        raise ValueError(f"{what}: tensor must be contiguous")
    if dtype is not None and str(t.dtype) != "torch." + dtype:
        raise TypeError(f"{what}: expected {dtype}, got {t.dtype}")
    if device is not None and t.device.type != device:
        raise TypeError(f"{what}: expected a {device} tensor, got {t.device}")
    if numel is not None and t.numel() < numel:
        raise ValueError(f"{what}: {t.numel()} elements, need {numel}")
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return C.c_void_p(stream)
    return C.c_void_p(stream.cuda_stream)


def opt_defaults(**kw) -> CsOpt:
    o = CsOpt()
    lib().cs_opt_defaults(C.byref(o))
    for k, v in kw.items():
        setattr(o, k, v)
    return o


def spherical_kmeans(vecs, K, cent, labels, iters=10, region=None, prob_region=None, stream=None):
    """cs_spherical_kmeans: vecs float64 cuda [npix,3]; K host int32 [nprob]; cent float64 cuda [sum K,3] (in: initial,
    out: final); labels int32 cuda [nprob,npix]; region uint8 cuda [npix] and prob_region host [nprob] or None."""
    K = np.ascontiguousarray(K, dtype=np.int32)
    nprob, npix = int(K.shape[0]), int(vecs.shape[0])
    if prob_region is not None:
        prob_region = np.ascontiguousarray(prob_region, dtype=np.int32)
    _chk(lib().cs_spherical_kmeans(npix, _ptr(vecs, "float64", "cuda", 3 * npix, "vecs"), _ptr(region, "uint8", "cuda", npix, "region"),
                                   nprob, _hp(K), _hp(prob_region), _ptr(cent, "float64", "cuda", 3 * int(K.sum()), "cent"), int(iters),
                                   _ptr(labels, "int32", "cuda", nprob * npix, "labels"), _stream(stream)), "cs_spherical_kmeans")


def spherical_kmeans_static(vecs, K, cent, labels, iters=10, region=None, prob_region=None, stream=None):
    """cs_spherical_kmeans_static: same arguments and same bits as spherical_kmeans, for a caller that must not allocate
    device memory (its pool owns the whole GPU, or it cannot afford the synchronisation an allocation may bring).  The
    library's only scratch, the table of problem descriptors, sits in a fixed 16-KiB device array shared by all calls:
    at most KMEANS_STATIC_MAX_PROB problems per call (CsError ELIMIT beyond), calls that may overlap on the GPU must be
    serialised by the caller, and the first call on a device should come before any stream capture."""
    K = np.ascontiguousarray(K, dtype=np.int32)
    nprob, npix = int(K.shape[0]), int(vecs.shape[0])
    if prob_region is not None:
        prob_region = np.ascontiguousarray(prob_region, dtype=np.int32)
    _chk(lib().cs_spherical_kmeans_static(npix, _ptr(vecs, "float64", "cuda", 3 * npix, "vecs"), _ptr(region, "uint8", "cuda", npix, "region"),
                                          nprob, _hp(K), _hp(prob_region), _ptr(cent, "float64", "cuda", 3 * int(K.sum()), "cent"), int(iters),
                                          _ptr(labels, "int32", "cuda", nprob * npix, "labels"), _stream(stream)), "cs_spherical_kmeans_static")


class Context:
    """Owns a cs_ctx*.  Methods mirror the C calls one to one (cs_<name> -> <name>)."""

    def __init__(self, freqs_ghz, npix, nu0_dust=353.0, nu0_sync=23.0, t_cmb=2.7255, units=UNITS_KCMB, options=None):
        self._freqs = np.ascontiguousarray(freqs_ghz, dtype=np.float64)
        m = CsModel(len(self._freqs), self._freqs.ctypes.data_as(C.POINTER(C.c_double)), float(nu0_dust),
                    float(nu0_sync), float(t_cmb), int(units), int(npix))
        self._h = C.c_void_p()
        self.nfreq, self.npix = len(self._freqs), int(npix)
        self.batch = 0
        self.nregion = 1
        self._keep = {}
        self.nparam = 0
        _chk(lib().cs_create(C.byref(self._h), C.byref(m)), "cs_create")
        for key, value in (options or {}).items():
            self.set_option(key, value)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().cs_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key, value):
        """key: OPT_* or one of "layout", "form", "min_fill", "copy_limit_mb"."""
        names = {"layout": OPT_LAYOUT, "form": OPT_FORM, "min_fill": OPT_MIN_FILL, "copy_limit_mb": OPT_COPY_LIMIT_MB,
                 "pixel_beta": OPT_PIXEL_BETA}
        _chk(lib().cs_set_option(self._h, int(names.get(key, key)), float(value)), "cs_set_option")

    def layout_info(self, cfg):
        """(sorted, ntile, fill) of configuration cfg."""
        so, nt, fill = C.c_int32(), C.c_int32(), C.c_double()
        _chk(lib().cs_layout_info(self._h, int(cfg), C.byref(so), C.byref(nt), C.byref(fill)), "cs_layout_info")
        return bool(so.value), nt.value, fill.value

    def model_constants(self):
        """dict(cd, cs, lnd, lns [nfreq], inv_sum_w): the host-computed constants the kernels are given."""
        arr = {k: np.empty(self.nfreq) for k in ("cd", "cs", "lnd", "lns")}
        inv = C.c_double()
        _chk(lib().cs_model_constants(self._h, _hp(arr["cd"]), _hp(arr["cs"]), _hp(arr["lnd"]), _hp(arr["lns"]), C.byref(inv)),
             "cs_model_constants")
        arr["inv_sum_w"] = inv.value
        return arr

    def set_clusters(self, maps, Kmap, cfg_maps, region_idx=None, nregion=1):
        """maps: int32 [nmap,npix] (torch device tensor or numpy); Kmap, cfg_maps: host arrays."""
        Kmap = np.ascontiguousarray(Kmap, dtype=np.int32)
        cfg_maps = np.ascontiguousarray(cfg_maps, dtype=np.int32).reshape(-1, 3)
        nmap = int(Kmap.shape[0])
        _chk(lib().cs_set_clusters(self._h, nmap, _ptr(maps, "int32", numel=nmap * self.npix, what="maps"), _hp(Kmap),
                                   int(cfg_maps.shape[0]), _hp(cfg_maps),
                                   _ptr(region_idx, "uint8", numel=self.npix, what="region_idx"), int(nregion)), "cs_set_clusters")
        self.nregion = int(nregion)
        self.batch = 0

    def set_data(self, d, ninv):
        """d: float32 device tensor [ndata,nfreq,2,npix] (borrowed: kept alive here); ninv: [nfreq] float32."""
        ndata = int(d.shape[0])
        if isinstance(ninv, np.ndarray):
            ninv = np.ascontiguousarray(ninv, dtype=np.float32)
        _chk(lib().cs_set_data(self._h, ndata, _ptr(d, "float32", "cuda", ndata * self.nfreq * 2 * self.npix, "d"),
                               _ptr(ninv, "float32", numel=self.nfreq, what="ninv")), "cs_set_data")
        self._keep["d"] = d

    def set_batch(self, cfg_of, data_of):
        cfg_of = np.ascontiguousarray(cfg_of, dtype=np.int32)
        data_of = np.ascontiguousarray(data_of, dtype=np.int32)
        _chk(lib().cs_set_batch(self._h, int(cfg_of.shape[0]), _hp(cfg_of), _hp(data_of)), "cs_set_batch")
        self.batch = int(cfg_of.shape[0])
        self.nparam = int(self.param_offsets()[-1])

    def param_offsets(self):
        off = np.empty(self.batch + 1, dtype=np.int64)
        _chk(lib().cs_param_offsets(self._h, _hp(off)), "cs_param_offsets")
        return off

    def build_sed_tables(self, params, stream=None):
        _chk(lib().cs_build_sed_tables(self._h, _ptr(params, "float64", "cuda", self.nparam, "params"), _stream(stream)),
             "cs_build_sed_tables")

    def spectral_like_grad(self, nll, grad=None, stream=None):
        _chk(lib().cs_spectral_like_grad(self._h, _ptr(nll, "float64", "cuda", self.batch * self.nregion, "nll"),
                                         _ptr(grad, "float64", "cuda", self.nparam, "grad"), _stream(stream)), "cs_spectral_like_grad")

    def spectral_misfit(self, chi2, stream=None):
        _chk(lib().cs_spectral_misfit(self._h, _ptr(chi2, "float64", "cuda", self.batch * self.nregion, "chi2"), _stream(stream)),
             "cs_spectral_misfit")

    def cell_moments(self, stream=None):
        _chk(lib().cs_cell_moments(self._h, _stream(stream)), "cs_cell_moments")

    def spectral_like_grad_cells(self, nll, grad=None, stream=None):
        _chk(lib().cs_spectral_like_grad_cells(self._h, _ptr(nll, "float64", "cuda", self.batch * self.nregion, "nll"),
                                               _ptr(grad, "float64", "cuda", self.nparam, "grad"), _stream(stream)),
             "cs_spectral_like_grad_cells")

    def component_maps(self, s, entries=None, stream=None):
        if entries is None:
            nsel, ep = self.batch, None
        else:
            entries = np.ascontiguousarray(entries, dtype=np.int32)
            nsel, ep = int(entries.shape[0]), _hp(entries)
        _chk(lib().cs_component_maps(self._h, nsel, ep, _ptr(s, "float32", "cuda", nsel * 6 * self.npix, "s"), _stream(stream)),
             "cs_component_maps")

    def cmb_residual_maps(self, cmb, data_sel, entries=None, stream=None):
        """cmb: float32 device [nsel,2,npix]; data_sel: data set each selected entry's W is applied to."""
        data_sel = np.ascontiguousarray(data_sel, dtype=np.int32)
        nsel = int(data_sel.shape[0])
        ep = None
        if entries is not None:
            entries = np.ascontiguousarray(entries, dtype=np.int32)
            assert entries.shape[0] == nsel
            ep = _hp(entries)
        _chk(lib().cs_cmb_residual_maps(self._h, nsel, ep, _hp(data_sel), _ptr(cmb, "float32", "cuda", nsel * 2 * self.npix, "cmb"),
                                        _stream(stream)), "cs_cmb_residual_maps")

    def cmb_variance(self, var, stream=None):
        _chk(lib().cs_cmb_variance(self._h, _ptr(var, "float64", "cuda", self.batch * self.nregion, "var"), _stream(stream)),
             "cs_cmb_variance")

    def optimize(self, params, lower, upper, opt=None, nll_final=None, stream=None):
        opt = opt or opt_defaults()
        n = self.nparam
        _chk(lib().cs_optimize(self._h, _ptr(params, "float64", "cuda", n, "params"), _ptr(lower, "float64", "cuda", n, "lower"),
                               _ptr(upper, "float64", "cuda", n, "upper"), C.byref(opt),
                               _ptr(nll_final, "float64", "cuda", self.batch, "nll_final"), _stream(stream)), "cs_optimize")

    def eval_host(self, d_host, ninv_host, params_host, nll_host, grad_host=None):
        """Host buffers in, host buffers out (numpy arrays or pinned torch CPU tensors)."""
        ndata = int(d_host.shape[0])
        _chk(lib().cs_eval_host(self._h, ndata, _ptr(d_host, "float32", "cpu", ndata * self.nfreq * 2 * self.npix, "d_host"),
                                _ptr(ninv_host, "float32", "cpu", self.nfreq, "ninv_host"),
                                _ptr(params_host, "float64", "cpu", self.nparam, "params_host"),
                                _ptr(nll_host, "float64", "cpu", self.batch * self.nregion, "nll_host"),
                                _ptr(grad_host, "float64", "cpu", self.nparam, "grad_host")), "cs_eval_host")

    def check(self, stream=None):
        return lib().cs_check(self._h, _stream(stream))

    def profile(self, enable=True):
        _chk(lib().cs_profile(self._h, 1 if enable else 0), "cs_profile")

    def profile_read(self):
        """(total ms, launches) of the fused gradient kernel since profile(True)."""
        ms, n = C.c_double(), C.c_int64()
        _chk(lib().cs_profile_read(self._h, C.byref(ms), C.byref(n)), "cs_profile_read")
        return ms.value, n.value

    def workspace_bytes(self):
        return int(lib().cs_workspace_bytes(self._h))

    def kernel_launches(self):
        return int(lib().cs_kernel_launches(self._h))
