"""B200-native calibrate + HEALPix-resample hot path of Argus-HDPS (arXiv 2207.14304).

The product is the C-ABI library ``libargus.so`` (include/argus.h, csrc/); this package is a thin ctypes
binding with the same entry-point names.  There is no CPU fallback: importing :mod:`binding` without the
compiled library raises.
"""
from .binding import (  # noqa: F401
    ARGUS_BILINEAR,
    ARGUS_LANCZOS3,
    ArgusError,
    Context,
    SOURCE_DTYPE,
    TRANSIENT_DTYPE,
    argus_background_map,
    argus_background_map_static,
    argus_calibrate,
    argus_coadd_accumulate,
    argus_detect_frame,
    argus_detect_frame_info,
    argus_detect_sources,
    argus_healpix_footprint,
    argus_plan_info,
    argus_prepare_masters,
    argus_resample,
    argus_resample_coadd,
    argus_resample_host,
    argus_resample_coadd_host,
    argus_reduce_frame_host,
    argus_host_wait,
    argus_segment_products,
    argus_subtract_tiles,
    library_path,
    load_library,
)
