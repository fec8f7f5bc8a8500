"""paper_2501_03322_b200 -- B200-native finite-source binary-lens magnification by contour integration
(the hot path of arXiv 2501.03322, "Twinkle").  The product is csrc/ (CUDA, sm_100a) behind the C ABI of
include/twk.h; this package is the thin Python binding (argument marshalling only).  There is no CPU fallback:
every compute entry point raises if libtwk.so or a CUDA device is missing."""
from .binding import (TWK_ST_CAP, TWK_ST_CONVERGED, TWK_ST_DOMAIN, TWK_ST_NUMERIC, TWK_ST_POINT, TWK_ST_REPAIRED, TWK_ST_SLOPE, Context, TwkError,
                      exported_symbols, lib, library_path, twk_debug_counters, twk_fp64_peak_probe, twk_magnify_static, twk_version, twk_workspace_bytes,
                      TWK_ELIMIT, TWK_STATIC_MAX_SOURCES)

__all__ = ["Context", "TwkError", "lib", "library_path", "exported_symbols", "twk_workspace_bytes", "twk_version",
           "twk_fp64_peak_probe", "twk_debug_counters", "twk_magnify_static", "TWK_STATIC_MAX_SOURCES", "TWK_ELIMIT", "TWK_ST_CONVERGED", "TWK_ST_CAP", "TWK_ST_REPAIRED", "TWK_ST_DOMAIN", "TWK_ST_NUMERIC", "TWK_ST_SLOPE", "TWK_ST_POINT"]
