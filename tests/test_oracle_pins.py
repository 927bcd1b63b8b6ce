"""Pins for the CPU oracle (oracle/etx_oracle.cpp): closed forms, brute force, library routines
and invariants, chosen so that a plausible mistake anywhere in it fails one of them.
The paper prints no worked numerical example, so nothing here is a number
printed by the paper; each test cites the passage whose definition it checks.  CPU only."""
import math

import numpy as np
import pytest
import torch

import datagen
import oracle
from helpers import (check_edge_invariants, check_track_invariants, components_bfs,
                     components_paper_sweeps, d2_exact_f32, knn_bruteforce, knn_replace_the_max,
                     set_layer, toy_config, zero_layers)

F = np.float32


# ------------------------------------------------------------------ features (L107 fn.5; R1)
def test_features_closed_form_and_true_division():
    cfg = toy_config()
    o = oracle.Oracle(datagen.pack_blob(cfg, zero_layers(cfg)))
    xyz = np.array([[40, -40, -300], [20, 10, 750], [0, 0, 225]], F)
    f = o.features(xyz)
    assert np.array_equal(f, np.array([[1, -1, 0], [0.5, 0.25, 1], [0, 0, 0.5]], F))
    rng = np.random.default_rng(1)
    xyz = rng.uniform(-60, 60, (4000, 3)).astype(F)
    xyz[:, 2] = rng.uniform(-300, 800, 4000)
    want = (xyz + np.array([0, 0, 300], F)) / np.array([40, 40, 1050], F)   # numpy fp32: IEEE add, divide
    assert np.array_equal(o.features(xyz), want)
    # a reciprocal multiply would differ somewhere: make sure this batch can tell
    recip = (xyz + np.array([0, 0, 300], F)) * (F(1) / np.array([40, 40, 1050], F))
    assert not np.array_equal(recip, want)


# ------------------------------------------------------------------ MLP forward (L96; R3)
def _emb_toy(D=4, H=2):
    cfg = toy_config(D=D, H=H)
    return cfg, zero_layers(cfg)


def test_embedding_selector_weights_closed_form():
    cfg, L = _emb_toy(D=4, H=2)
    # layer0 picks (fx, fy, fz, -fx); ReLU kills negatives; layer1 identity; last layer sums pairs
    set_layer(L, "emb0", [[1, 0, 0], [0, 1, 0], [0, 0, 1], [-1, 0, 0]], [0, 0, 0, 0])
    set_layer(L, "emb1", np.eye(4), [0, 0, 0, 0.5])
    set_layer(L, "emb2", [[1, 1, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1], [1, 1, 1, 1]], [0, 0, 0, -1])
    o = oracle.Oracle(datagen.pack_blob(cfg, L))
    xyz = np.array([[20, 10, 225], [-20, 30, -300], [10, -10, 750]], F)   # f = (.5,.25,.5), (-.5,.75,0), (.25,-.25,1)
    want = np.array([[0.75, 0.5, 0.5, 0.75 + 0.5 + 0.5 - 1],
                     [0.75, 0.0, 1.0, 0.75 + 0 + 1.0 - 1],              # relu(-0.5)=0 ; relu(+0.5)+0.5 = 1.0
                     [0.25, 1.0, 0.5, 0.25 + 1.0 + 0.5 - 1]], F)        # relu(-.25)=0
    assert np.array_equal(o.embed(xyz), want)


def test_embedding_no_relu_on_output_and_bias_everywhere():
    cfg, L = _emb_toy(D=4, H=1)
    set_layer(L, "emb0", np.zeros((4, 3)), [1, 2, -3, 4])            # hidden = relu(b) = (1,2,0,4)
    set_layer(L, "emb1", -np.eye(4), [0.5, 0.5, 0.5, 0.5])           # out = -hidden + .5 (negative kept)
    o = oracle.Oracle(datagen.pack_blob(cfg, L))
    assert np.array_equal(o.embed(np.zeros((2, 3), F)), np.tile(np.array([-0.5, -1.5, 0.5, -3.5], F), (2, 1)))


def test_embedding_matches_float64_matmul_within_bound():
    cfg = datagen.get_config("cfg1")
    W = datagen.make_weights(cfg, "parity")
    o = oracle.Oracle(datagen.pack_blob(cfg, W))
    b = datagen.generate_batch(cfg, n_events=1)
    got = o.embed(b.xyz).astype(np.float64)
    x = o.features(b.xyz).astype(np.float64)
    bound = np.zeros(x.shape[0])
    H = cfg.emb_n_hidden_layers
    for li in range(H + 1):
        _, Wl, bl = W[li]
        mag = np.abs(x) @ np.abs(Wl.T.astype(np.float64)) + np.abs(bl)
        x = x @ Wl.T.astype(np.float64) + bl
        if li < H:
            x = np.maximum(x, 0)
        bound = bound * np.abs(Wl).sum(1).max() + (Wl.shape[1] + 1) * 2.0 ** -24 * mag.max(1)
    err = np.abs(got - x).max(1)
    assert np.all(err <= bound + 1e-12)
    assert err.max() > 0          # it really is fp32, not a float64 computation in disguise
    assert err.max() < 1e-4


def test_pinned_accumulation_order_ascending_j():
    # acc = fma(x_j, w_j, acc) for j ascending from acc = 0, then + b (R3/R4).  With products
    # (2^24, 1, 1) and b = -2^24: ascending gives ((2^24 + 1 -> 2^24, tie to even) + 1 -> 2^24) + b = 0;
    # descending gives (1 + 1) + 2^24 = 2^24 + 2, + b = 2; bias-first gives 2 as well.
    cfg, L = _emb_toy(D=4, H=1)
    set_layer(L, "emb0", [[1, 0, 0], [0, 1, 0], [0, 0, 1], [0, 0, 0]])
    set_layer(L, "emb1", [[2.0 ** 24, 1, 1, 0], [1, 1, 2.0 ** 24, 0], [0, 0, 0, 0], [0, 0, 0, 0]],
              [-(2.0 ** 24), -(2.0 ** 24), 0, 0])
    o = oracle.Oracle(datagen.pack_blob(cfg, L))
    out = o.embed(np.array([[40, 40, 750]], F))      # f = (1, 1, 1): hidden = (1, 1, 1, 0)
    assert out[0, 0] == 0.0
    assert out[0, 1] == 2.0                          # same numbers, big term last: (1 + 1) + 2^24 exact


# ------------------------------------------------------------------ bf16 rounding (R20)
def test_bf16_round_matches_torch_on_all_upper_halves_and_ties():
    hi = np.arange(0, 1 << 16, dtype=np.uint32) << 16
    lows = np.array([0x0000, 0x0001, 0x7FFF, 0x8000, 0x8001, 0xFFFF], np.uint32)
    bits = (hi[:, None] | lows[None, :]).reshape(-1)
    x = bits.view(np.float32)
    finite = np.isfinite(x)
    want = torch.from_numpy(x.copy()).to(torch.bfloat16).to(torch.float32).numpy()
    got = np.array([oracle.bf16_round(float(v)) for v in x[finite][::7]], F)
    assert np.array_equal(got.view(np.uint32), want[finite][::7].view(np.uint32))
    # explicit ties: 1 + 2^-8 is halfway between 1 and 1+2^-7 -> even (1.0); 1 + 3*2^-8 -> 1 + 2^-6
    assert oracle.bf16_round(1 + 2.0 ** -8) == 1.0
    assert oracle.bf16_round(1 + 3 * 2.0 ** -8) == 1 + 2.0 ** -6
    assert math.isinf(oracle.bf16_round(float("inf")))


def test_bf16_mode_rounds_weights_and_hidden_activations_not_output():
    cfg, L = _emb_toy(D=16, H=2)
    w = 1 + 2.0 ** -9                                   # not a bf16 number: rounds to 1.0
    W0 = np.zeros((16, 3)); W0[0, 0] = 1.0
    set_layer(L, "emb0", W0)                            # K=3 layer stays fp32 (R20)
    W1 = np.zeros((16, 16)); W1[0, 0] = w
    set_layer(L, "emb1", W1)
    W2 = np.zeros((4, 16)); W2[0, 0] = 1.0
    set_layer(L, "emb2", W2, [2.0 ** -12, 0, 0, 0])
    blob = datagen.pack_blob(cfg, L)
    x = np.array([[40 * (1 + 2.0 ** -10), 0, 0]], F)    # f_x = 1+2^-10 exactly representable in fp32 only
    fx = oracle.Oracle(blob, "fp32").features(x)[0, 0]
    o32 = oracle.Oracle(blob, "fp32").embed(x)[0, 0]
    o16 = oracle.Oracle(blob, "bf16").embed(x)[0, 0]
    assert o32 == F(F(fx) * F(w)) + F(2.0 ** -12)
    # bf16: hidden0 = bf16(fx) = 1.0; W1 -> 1.0; hidden1 = 1.0; output = 1 + 2^-12 kept in fp32
    assert o16 == F(1.0) + F(2.0 ** -12)


# ------------------------------------------------------------------ int8 (R21)
def test_int8_quantiser_hand_values():
    q = oracle.quant_i8
    assert q(0.0, 1.0) == 0 and q(1.0, 1.0) == 1 and q(-1.0, 1.0) == -1
    assert q(0.5, 1.0) == 0 and q(1.5, 1.0) == 2 and q(2.5, 1.0) == 2 and q(-0.5, 1.0) == 0 and q(-1.5, 1.0) == -2
    assert q(1000.0, 1.0) == 127 and q(-1000.0, 1.0) == -127 and q(-127.6, 1.0) == -127
    assert q(1.0, 0.5) == 2 and q(63.4, 0.5) == 127


def test_int8_layer_accumulators_equal_integer_matmul():
    cfg = datagen.get_config("cfg0")
    W = datagen.make_weights(cfg, "parity")
    b = datagen.generate_batch(cfg)
    scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window)
    assert scales.size == datagen.n_act_scales(cfg) and np.all(scales > 0)
    blob = datagen.pack_blob(cfg, W, scales)
    o = oracle.Oracle(blob, "int8")
    names = [n for n, _, _ in datagen.layer_shapes(cfg)]
    li = names.index("emb1")                              # 64 -> 64, input = relu(emb0(f)) in fp32
    tap = np.zeros((b.n_hits, 64), np.int32)
    o.set_tap(li, tap)
    emb = o.embed(b.xyz)
    o.set_tap(-1, None)
    Wq, sw, sx = o.qweights(li, 64, 64)
    # independent: numpy fp32 layer 0, numpy quantiser, int64 matmul
    f = oracle.Oracle(blob, "fp32").features(b.xyz)
    _, W0, b0 = W[0]
    h0 = np.maximum(_fma_chain(f, W0) + b0, 0).astype(F)
    inv = F(1.0) / F(sx)
    qx = np.clip(np.rint(h0 * inv), -127, 127).astype(np.int64)
    assert np.array_equal(tap.astype(np.int64), qx @ Wq.astype(np.int64).T)
    # per-channel weight scales and quantised weights (max|w|/127, rne, clamp)
    _, W1, _ = W[li]
    assert np.array_equal(sw, (np.abs(W1).max(1) / F(127)).astype(F))
    assert np.array_equal(Wq, np.clip(np.rint(W1 / sw[:, None]), -127, 127).astype(np.int8))
    assert np.abs(Wq).max() == 127
    assert np.isfinite(emb).all()


def _fma_chain(x, W):
    """fp32 fma chain over ascending j, emulated exactly in float64 for K=3 (each step: one rounding)."""
    acc = np.zeros((x.shape[0], W.shape[0]), F)
    for j in range(W.shape[1]):
        acc = (x[:, j:j + 1].astype(np.float64) * W[None, :, j].astype(np.float64) + acc.astype(np.float64)).astype(F)
    return acc
