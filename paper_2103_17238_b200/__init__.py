"""paper_2103_17238_b200 -- B200-native Super-Droplet Method coalescence step.

Thin Python binding over the C-ABI library `libsdm_b200.so` (include/sdm.h).  It only marshals
arguments: every step of the hot path runs in the hand-written sm_100a kernels under csrc/.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback: without
the built CUDA library, or without a CUDA device, the calls raise.
"""
from .binding import (  # noqa: F401
    GEOMETRIC,
    GEOMETRIC_TABLE,
    GOLOVIN,
    PATH_AUTO,
    PATH_CELL_SORTED,
    PATH_GENERAL,
    PATH_HYBRID,
    PATH_BOX,
    PATH_BUCKET,
    OPT_NARROW_KEY_BITS,
    OPT_TRACK_ZEROS,
    OPT_INDEX_BASE,
    OPT_SKIP_KEY_DIGITS,
    OPT_FUSED_WORDS_PER_LANE,
    OPT_BUCKET_BITS,
    OPT_BOX_CLUSTER,
    KernelParams,
    SDMContext,
    SDMError,
    geometric,
    geometric_table,
    golovin,
    host_staging_bytes,
    library_path,
    load_library,
    remove_zero_multiplicity_static,
    static_max_n_sd,
    workspace_bytes,
)

__all__ = [
    "SDMContext", "SDMError", "KernelParams", "golovin", "geometric", "geometric_table", "GOLOVIN", "GEOMETRIC", "GEOMETRIC_TABLE",
    "PATH_AUTO", "PATH_GENERAL", "PATH_CELL_SORTED", "PATH_HYBRID", "PATH_BOX", "PATH_BUCKET", "OPT_NARROW_KEY_BITS", "OPT_TRACK_ZEROS", "OPT_INDEX_BASE", "OPT_SKIP_KEY_DIGITS", "OPT_FUSED_WORDS_PER_LANE", "OPT_BUCKET_BITS", "OPT_BOX_CLUSTER", "workspace_bytes", "host_staging_bytes",
    "load_library", "library_path", "remove_zero_multiplicity_static", "static_max_n_sd",
]
