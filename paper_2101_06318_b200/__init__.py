"""B200-native Super-Droplet Method coalescence step (arXiv 2101.06318) behind a C ABI.

``libsdm.so`` (hand-written CUDA for sm_100a, see ``csrc/`` and ``include/sdm.h``) does all the
work; this package is a thin ctypes binding with the same call names.  PyTorch supplies device
memory and the CUDA stream only.  There is no CPU fallback: if the library is not built or no
CUDA device is present, calls raise.
"""
from .binding import (  # noqa: F401
    SDM,
    SdmError,
    KERNEL_GOLOVIN,
    KERNEL_GRAVITATIONAL,
    KERNEL_GRAVITATIONAL_TABULATED,
    KERNEL_USER,
    OPT_FORCE_GENERAL,
    OPT_SEGMENT_CAP,
    OPT_WRITE_IDX,
    OPT_SCREENING,
    OPT_TIMING,
    OPT_LANES_PER_CELL,
    OPT_SORT_ENGINE,
    OPT_DETERMINISTIC,
    OPT_CTAS_PER_SM,
    OPT_BOX_CTAS,
    OPT_BOX_REGION_CAP,
    OPT_BOX_SORT_CAP,
    OPT_COOPERATIVE,
    load_library,
    library_path,
    workspace_bytes,
    version,
    moments_noalloc,
    NOALLOC_MAX_SD,
)
