"""Seeded random weights and the weights-blob container (layout: include/etx.h).

No method arithmetic: this draws numbers and packs bytes.  bf16 / int8
conversion of weights is done separately inside the oracle and inside
`etx_create`, each from these same fp32 bytes.

Blob (little-endian):
  header, 16 x uint32:
    [0] magic 'ETXW' (0x57585445)  [1] version = 1
    [2] emb_hidden  [3] emb_n_hidden_layers  [4] emb_dim
    [5] gnn_latent  [6] gnn_iters            [7] edge_enc_input
    [8] n_weight_floats  [9] n_act_scales    [10] emb_input   [11] triplet classifiers present
    [12..15] zero
  then fp32 tensors, each Linear as W[out][in] row-major followed by b[out], in
  this order: embedding layers 0..H; node encoder (2); edge encoder (2); for each
  iteration: node net (2), edge net (2); head (1); with word 11 set, the
  articulation classifier (2d -> d, d -> 1) and the elbow classifier (same
  shapes).  Concatenated inputs are ordered [h, m_out, m_in], [h_src, h_dst, e]
  and [e_first, e_second].
  then n_act_scales fp32 activation scales (INT8 only; one per quantised Linear,
  in layer order).
"""
from __future__ import annotations

import math
import struct

import numpy as np

from .configs import EtxConfig

BLOB_MAGIC = 0x57585445
BLOB_VERSION = 1
HEADER_WORDS = 16


def layer_shapes(cfg: EtxConfig) -> list[tuple[str, int, int]]:
    """[(name, out, in)] in blob order."""
    D, H, nd, d, L = cfg.emb_hidden, cfg.emb_n_hidden_layers, cfg.emb_dim, cfg.gnn_latent, cfg.gnn_iters
    out: list[tuple[str, int, int]] = [("emb0", D, 3)]
    for i in range(1, H):
        out.append((f"emb{i}", D, D))
    out.append((f"emb{H}", nd, D))
    out += [("nenc0", d, 3), ("nenc1", d, d)]
    kee = 3 if cfg.edge_enc_input == 0 else 2 * d
    out += [("eenc0", d, kee), ("eenc1", d, d)]
    for it in range(L):
        out += [(f"node{it}_0", d, 3 * d), (f"node{it}_1", d, d),
                (f"edge{it}_0", d, 3 * d), (f"edge{it}_1", d, d)]
    out.append(("head", 1, d))
    if getattr(cfg, "triplets", 0):           # articulation and elbow classifiers on [e_first, e_second] (L80, L160)
        out += [("tart0", d, 2 * d), ("tart1", 1, d), ("telb0", d, 2 * d), ("telb1", 1, d)]
    return out


def quantised_layer_names(cfg: EtxConfig) -> list[str]:
    """Linears that are quantised in INT8 mode: every Linear with in >= 16 except the
    d->1 head (reading R21), in blob order."""
    return [n for (n, o, i) in layer_shapes(cfg) if i >= 16 and n not in ("head", "tart1", "telb1")]


def n_act_scales(cfg: EtxConfig) -> int:
    return len(quantised_layer_names(cfg))


def make_weights(cfg: EtxConfig, preset: str = "he", seed: int | None = None
                 ) -> list[tuple[str, np.ndarray, np.ndarray]]:
    """[(name, W[out][in] fp32, b[out] fp32)] in blob order.

    preset "he":     He-uniform U(+-sqrt(6/fan_in)), zero biases (BASELINE.json configs).
    preset "parity": same draw, then tamed so that activations stay O(1) and logits
                     spread around 0: message columns of each node
                     net's first layer / (2k), last layer of each node/edge net x 0.25,
                     biases U(+-0.1), head weights x 2.  Exercises the bias
                     path and keeps scores away from 0/1 so score parity is informative.
    """
    seed = cfg.weights_seed if seed is None else seed
    rng = np.random.Generator(np.random.Philox(key=[seed, 0xE7]))
    layers = []
    d = cfg.gnn_latent
    for (name, o, i) in layer_shapes(cfg):
        bound = math.sqrt(6.0 / i)
        W = rng.uniform(-bound, bound, (o, i)).astype(np.float32)
        bdraw = rng.uniform(-0.1, 0.1, o).astype(np.float32)      # drawn always: same stream for both presets
        b = np.zeros(o, np.float32)
        if preset == "parity":
            b = bdraw
            if name.startswith("node") and name.endswith("_0"):
                W[:, d:] *= np.float32(1.0 / (2.0 * cfg.k))
            if (name.startswith("node") or name.startswith("edge")) and name.endswith("_1"):
                W *= np.float32(0.25)
            if name in ("head", "tart1", "telb1"):
                W *= np.float32(2.0)
        elif preset != "he":
            raise ValueError(preset)
        layers.append((name, W, b))
    return layers


def pack_blob(cfg: EtxConfig, layers, act_scales: np.ndarray | None = None) -> bytes:
    shapes = layer_shapes(cfg)
    assert [s[0] for s in shapes] == [l[0] for l in layers]
    parts = []
    for (name, o, i), (_, W, b) in zip(shapes, layers):
        assert W.shape == (o, i) and b.shape == (o,), name
        parts.append(np.ascontiguousarray(W, dtype="<f4").tobytes())
        parts.append(np.ascontiguousarray(b, dtype="<f4").tobytes())
    body = b"".join(parts)
    n_floats = len(body) // 4
    sc = np.zeros(0, "<f4") if act_scales is None else np.ascontiguousarray(act_scales, dtype="<f4")
    hdr = [BLOB_MAGIC, BLOB_VERSION, cfg.emb_hidden, cfg.emb_n_hidden_layers, cfg.emb_dim,
           cfg.gnn_latent, cfg.gnn_iters, cfg.edge_enc_input, n_floats, int(sc.size), cfg.emb_input,
           int(getattr(cfg, "triplets", 0))] + [0] * 4
    return struct.pack("<16I", *hdr) + body + sc.tobytes()


def unpack_blob(cfg: EtxConfig, blob: bytes):
    """Inverse of pack_blob (for tests that need the raw matrices)."""
    hdr = struct.unpack("<16I", blob[:64])
    assert hdr[0] == BLOB_MAGIC and hdr[1] == BLOB_VERSION
    arr = np.frombuffer(blob, dtype="<f4", offset=64)
    pos, layers = 0, []
    for (name, o, i) in layer_shapes(cfg):
        W = arr[pos:pos + o * i].reshape(o, i).copy(); pos += o * i
        b = arr[pos:pos + o].copy(); pos += o
        layers.append((name, W, b))
    assert pos == hdr[8]
    scales = arr[pos:pos + hdr[9]].copy()
    return layers, scales
