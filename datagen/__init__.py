"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This package holds NONE of the method's arithmetic (no MLP, no k-NN, no
scatter, no components).  It only produces inputs: VELO-shaped events
(`velo.py`), random weights packed into the blob format of `include/etx.h`
(`weights.py`), and the hyper-parameter presets of BASELINE.json's five
configs (`configs.py`).  Recipe and citations: DESIGN.md section 5.
"""
from .configs import CONFIGS, EtxConfig, get_config  # noqa: F401
from .velo import generate_batch, EventBatch, hand_batch  # noqa: F401
from .weights import (make_weights, pack_blob, unpack_blob, layer_shapes,  # noqa: F401
                      n_act_scales, BLOB_MAGIC)
