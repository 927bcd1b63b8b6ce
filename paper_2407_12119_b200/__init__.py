"""paper_2407_12119_b200 -- B200-native ETX4VELO hot path (arXiv 2407.12119).

Thin ctypes binding of the C-ABI library `libetx.so` (include/etx.h): the same names, argument
marshalling only.  Every step of the path (embedding MLP, plane-restricted k-NN, edge compaction,
interaction-network edge classifier, threshold + connected components) runs in the library's CUDA
kernels; PyTorch is used only for device memory and streams.  There is no CPU fallback: using this
package without the built library, or without a CUDA device, raises.
"""
from .binding import (Etx, EtxError, EtxOutput, Hyperparams, Inject, STAGE_NAMES, hyperparams_from_config,  # noqa: F401
                      lib, lib_path, load_library, declared_symbols, tracks_static, TRACKS_STATIC_MAX_HITS)
