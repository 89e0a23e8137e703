"""B200-native DNN-SP2-PT hot path (arXiv 2203.09621): thin Python binding over the C ABI.

Every step of the path runs in the hand-written sm_100a kernels of `libdmpt.so`
(`csrc/`, C ABI in `include/dmpt.h`).  This package only marshals arguments; PyTorch supplies
device memory and streams.  There is no CPU fallback: importing `binding` without the built
library raises.
"""
from .binding import (  # noqa: F401
    Dmpt,
    DmptPair,
    DmptError,
    DmptOptions,
    DmptResult,
    dmpt_create,
    dmpt_default_options,
    dmpt_workspace_bytes_fields,
    dmpt_destroy,
    dmpt_last_cuda_error,
    dmpt_layer_products,
    dmpt_run,
    dmpt_run_host,
    dmpt_set_hamiltonian,
    dmpt_spectral_bounds,
    dmpt_spectral_bounds_noalloc,
    spectral_bounds_noalloc,
    dmpt_initial_transform,
    dmpt_split,
    dmpt_strerror,
    dmpt_workspace_bytes,
    lib,
    EXPORTED_SYMBOLS,
)
