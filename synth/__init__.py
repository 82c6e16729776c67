"""Seeded synthetic inputs shaped like the paper's IMX455 frames.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2207_14304_b200/``).  It holds none of the method's arithmetic
(no calibration, no HEALPix, no WCS projection, no interpolation): it only
draws raw frames, calibration masters and WCS parameters.

Recipe (Table 1 gives the detector:
61 MPix IMX455, 1.7 e- read noise, 1.38 arcsec/pix; BASELINE.json configs[0..4]
give the scene).  ``numpy.random.Generator(PCG64(seed))``; draws happen in this
fixed order: star x, star y, star flux quantile, flat noise, read noise,
photon counts, dark counts.
"""
from .frames import (  # noqa: F401
    Frame,
    Wcs,
    PIXEL_SCALE_DEG,
    make_wcs,
    make_sip,
    make_frame,
    inject_defects,
    config0,
    config1,
    config2_frame,
    config3_frame,
    config4_frame,
    special_pointings,
)
from .segments import footprint_like, target_list  # noqa: F401,E402
