"""B200-native Odyssey hot path (arXiv 1601.02063): Kerr null-geodesic integration fused with
general-relativistic radiative transfer, as hand-written sm_100a CUDA kernels behind a C ABI
(include/odyssey.h).  This package is the thin Python binding: argument marshalling only."""
from .binding import (  # noqa: F401
    OdysseyError, load_library, trace_geodesics, render_image, render_spectrum,
    trace_geodesics_host, render_image_host, render_spectrum_host, render_hotspot, render_hotspot_host,
    fp64_peak_probe, kernel_info, eval_math, PREC_FP64, PREC_MIXED_FP32, launch_count, trim_scratch, last_error, shutdown, EXPORTED_SYMBOLS,
)
