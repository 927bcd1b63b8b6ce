"""Seeded randomised parity campaign: the same comparisons as test_gpu_parity.py, over many seeds, event mixes and
model shapes.  By default a handful of seeds run with `pytest -m gpu`; ETX_CAMPAIGN=N widens every family to N seeds
(profiles/r2_campaign.md records one such run).  Every expected value comes from oracle/."""
import os

import numpy as np
import pytest
import torch

import datagen
import oracle
from gpu_utils import make_ctx, run_gpu, state
from helpers import centred_parity_weights

pytestmark = pytest.mark.gpu
F = np.float32
N = int(os.environ.get("ETX_CAMPAIGN", "3"))


def _random_case(seed, precision, triplets=0):
    rng = np.random.default_rng(9000 + seed)
    base = str(rng.choice(["cfg0", "cfg1", "cfg5"]))
    cfg = datagen.get_config(base).replace(precision=precision, triplets=triplets,
                                           k=int(rng.choice([3, 4, 8, 10, 16])), window=int(rng.integers(1, 4)),
                                           gnn_latent=int(rng.choice([32, 64])), gnn_iters=int(rng.integers(0, 4)),
                                           emb_hidden=int(rng.choice([64, 128])), emb_n_hidden_layers=int(rng.integers(1, 4)),
                                           edge_enc_input=int(rng.integers(0, 2)), d2_max=float(rng.choice([np.inf, np.inf, 0.5])),
                                           mu_pv=float(rng.choice([1.0, 3.0, 5.0])), events_seed=int(rng.integers(1, 1 << 20)))
    if precision == "int8":
        cfg = cfg.replace(state_dtype=str(rng.choice(["auto", "bf16"])))
    b = datagen.generate_batch(cfg, n_events=int(rng.integers(1, 5)))
    W = centred_parity_weights(cfg.replace(precision="fp32"), b, seed=int(rng.integers(1, 1000)))
    scales = None
    if precision == "int8":
        scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max)
    return cfg, b, datagen.pack_blob(cfg, W, scales)


@pytest.mark.parametrize("seed", range(N))
def test_campaign_fp32_end_to_end_bit_exact(seed):
    cfg, b, blob = _random_case(seed, "fp32")
    r = oracle.Oracle(blob, "fp32").run(b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    assert np.array_equal(g["emb"], r["emb"]), cfg
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"]), cfg
    assert np.array_equal(g["logit"], r["logit"]), cfg
    assert np.array_equal(g["track_id"], r["track_id"]), cfg
    ctx.destroy()


@pytest.mark.parametrize("seed", range(N))
def test_campaign_int8_end_to_end_bit_exact(seed):
    cfg, b, blob = _random_case(100 + seed, "int8")
    r = oracle.Oracle(blob, "int8", state_dtype=cfg.state_dtype).run(b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    assert np.array_equal(g["emb"], r["emb"]), cfg
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"]), cfg
    assert np.array_equal(g["logit"], r["logit"]), cfg
    assert np.array_equal(g["track_id"], r["track_id"]), cfg
    ctx.destroy()


@pytest.mark.parametrize("seed", range(N))
def test_campaign_bf16_chained_within_the_bar(seed):
    cfg, b, blob = _random_case(200 + seed, "bf16")
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    nbr, deg = oracle.knn(g["emb"], b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max)
    src, dst, _ = oracle.build_edges(nbr, deg)
    assert np.array_equal(g["src"], src) and np.array_equal(g["dst"], dst), cfg
    og = oracle.Oracle(blob, "bf16").gnn(b.xyz, src, dst)
    if src.size:
        assert np.abs(g["score"] - og["score"]).max() <= 2e-2, cfg
    tid = oracle.components(src, dst, g["logit"], oracle.logit_threshold(cfg.threshold), b.n_hits)
    assert np.array_equal(g["track_id"], tid), cfg
    ctx.destroy()


@pytest.mark.parametrize("seed", range(max(1, N // 2)))
def test_campaign_triplet_stage(seed):
    precision = ["fp32", "bf16", "int8"][seed % 3]
    cfg, b, blob = _random_case(300 + seed, precision, triplets=1)
    if cfg.gnn_iters == 0:
        cfg = cfg                                             # L = 0: the classifiers read the encoder output e^0
    ctx = make_ctx(cfg, blob, b, max_triplets=3_000_000)
    g = run_gpu(ctx, b, debug=False)
    E = g["n_edges"]
    t = ctx.triplets()
    keep = (g["logit"] >= oracle.logit_threshold(cfg.threshold)).astype(np.uint8)
    o = oracle.Oracle(blob, precision, state_dtype=cfg.state_dtype)
    e_gpu = state(ctx, "e", E, cfg.gnn_latent) if E else np.zeros((0, cfg.gnn_latent), F)
    tau_t = oracle.logit_threshold(cfg.triplet_threshold)
    pairs, kept = {}, {}
    for k, kind in enumerate(("articulation", "left_elbow", "right_elbow")):
        f, s, h = oracle.triplets(g["src"], g["dst"], keep, b.n_hits, kind)
        assert t["count"][k] == f.size <= 3_000_000, cfg
        assert np.array_equal(t[kind]["first"].cpu().numpy(), f) and np.array_equal(t[kind]["second"].cpu().numpy(), s), cfg
        z, sc = o.triplet_scores(e_gpu, f, s, elbow=(k > 0))
        gz = t[kind]["logit"].cpu().numpy()
        if precision == "bf16":
            assert np.abs(t[kind]["score"].cpu().numpy() - sc).max(initial=0) <= 2e-2, cfg
        else:
            assert np.array_equal(gz, z), cfg
        pairs[kind] = (f, s); kept[kind] = (gz >= tau_t).astype(np.uint8)
    tc = ctx.triplet_components(E)
    comp, shared = oracle.triplet_components(keep, pairs["articulation"], kept["articulation"], pairs["left_elbow"], kept["left_elbow"],
                                             pairs["right_elbow"], kept["right_elbow"])
    assert np.array_equal(tc["edge_component"].cpu().numpy(), comp), cfg
    got = tc["shared"].cpu().numpy()
    got = np.unique(got, axis=0) if got.size else got.reshape(0, 2)
    assert np.array_equal(got, shared), cfg
    # phases (3)-(4) in the product: the track list equals the oracle's four-phase result as arrays
    offs, hits = oracle.tracks_from_triplets(g["src"], g["dst"], keep, pairs["articulation"], kept["articulation"], pairs["left_elbow"],
                                             kept["left_elbow"], pairs["right_elbow"], kept["right_elbow"], 3)
    tt = ctx.triplet_tracks(3)
    assert tt["overflow"] == 0 and np.array_equal(tt["track_offsets"].cpu().numpy(), offs), cfg
    assert np.array_equal(tt["track_hits"].cpu().numpy(), hits), cfg
    ctx.destroy()
