"""B200 (sm_100a) sparse-sketch hot path: thin Python binding over the C-ABI library.

Every step of the path (hash, stream, sign/scale, convert, scatter-accumulate, flush) runs in the
CUDA kernels of ``csrc/``; this package only marshals arguments (``binding.py``).  There is no CPU
fallback: importing the binding raises if ``libsparse_sketch.so`` cannot be built or loaded.
"""
from .binding import (  # noqa: F401
    DITHER,
    RN,
    SR,
    VARIANT_AUTO,
    VARIANT_FLAT_PAIR,
    VARIANT_FLAT_VEC,
    VARIANT_GENERIC,
    VARIANT_SMEM,
    VARIANT_TMEM,
    VARIANT_SMALL,
    VARIANT_NAMES,
    Sketch,
    SketchError,
    SketchOpts,
    lib,
    library_path,
    sketch_convert_probe,
    sketch_launch_count,
    sketch_red_probe,
    sketch_stream_probe,
    sketch_strerror,
    sketch_widen,
    sketch_version,
)
