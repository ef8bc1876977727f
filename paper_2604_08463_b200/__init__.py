"""B200-native batched parametric spectral likelihood for CMB component separation (arxiv 2604.08463).

The product is the CUDA library `libcs.so` (C ABI: include/cs.h, sources: csrc/).  This package is its thin
Python binding; see DESIGN.md.
"""
from .binding import (  # noqa: F401
    Context, CsError, CsOpt, opt_defaults, lib, strerror, spherical_kmeans, spherical_kmeans_static, EXPORTS, ELIMIT, KMEANS_STATIC_MAX_PROB,
    OK, EINVAL, EINDEX, EDOMAIN, ESINGULAR, ECUDA, ENOMEM, UNITS_KCMB, UNITS_LITERAL,
    OPT_LAYOUT, OPT_FORM, OPT_MIN_FILL, OPT_COPY_LIMIT_MB, LAYOUT_AUTO, LAYOUT_INPLACE, LAYOUT_SORTED, FORM_AUTO, FORM_DIRECT, METHOD_ADATOPK, METHOD_LBFGS, OPT_PIXEL_BETA, PIXBETA_AUTO, PIXBETA_OFF,
)
