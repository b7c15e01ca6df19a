"""B200-native batched tree-physics step of OrchardBench (arxiv/paper_2607_06337).

The product is the C-ABI CUDA library `libob.so` (include/orchard.h, csrc/);
this package is its thin Python binding.  Nothing here imports `oracle/`.
"""
from .binding import (  # noqa: F401
    EXPORTS,
    LIB_PATH,
    OB_E_ARG,
    OB_E_CAPACITY,
    OB_E_CUDA,
    OB_E_WORKSPACE,
    OB_MAX_WRENCH,
    OB_OK,
    OB_STATUS_CG_MAXITER,
    OB_STATUS_NONFINITE,
    Orchard,
    OrchardError,
    default_params,
    load_library,
    marshal_specs,
    GEOMETRY_IDENTITY,
    ob_event,
    ob_geometry_ranges,
    ob_params,
    ob_world_spec,
    params_struct,
)
