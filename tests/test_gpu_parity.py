"""GPU parity: the CUDA path (through the C-ABI, via the ctypes binding) against the CPU oracle on identical
seeded inputs.  Protocol: DESIGN.md sec. 6 (stage-isolated, chained, end-to-end).  Bars (BASELINE.json
north_star): k-NN edge list and track ids bit-exact; scores within 1e-4 (fp32) / 2e-2 (bf16) absolute;
int32 accumulators of the INT8 path bit-exact."""
import numpy as np
import pytest
import torch

import datagen
import oracle
from gpu_utils import dev, make_ctx, run_gpu, state
from helpers import centred_parity_weights, check_edge_invariants, check_track_invariants

pytestmark = pytest.mark.gpu
F = np.float32


def _setup(name, n_events=None, preset="parity", precision=None, seed=None):
    cfg = datagen.get_config(name)
    if precision:
        cfg = cfg.replace(precision=precision)
    b = datagen.generate_batch(cfg, n_events=n_events, seed=seed)
    W = centred_parity_weights(cfg, b) if preset == "parity" else datagen.make_weights(cfg, preset)
    return cfg, b, W


def _oracle_all(cfg, b, blob, precision):
    o = oracle.Oracle(blob, precision, state_dtype=cfg.state_dtype)
    r = o.run(b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    r["col_ptr"], r["in_edge"] = oracle.csc(r["dst"], b.n_hits)
    return o, r


# ---------------------------------------------------------------------------------- S0 + S2 + S3
@pytest.mark.parametrize("name,n_events", [("cfg0", 1), ("cfg1", 5), ("cfg4", 2)])
def test_knn_and_edge_list_bit_exact_on_oracle_embedding(name, n_events):
    cfg, b, W = _setup(name, n_events, precision="fp32")
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "fp32")
    ctx = make_ctx(cfg, blob, b, precision="fp32")
    g = run_gpu(ctx, b, emb=r["emb"], last_stage=3)
    assert g["n_edges"] == r["src"].size
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"])
    assert np.array_equal(g["row_ptr"], r["row_ptr"])
    assert np.array_equal(g["col_ptr"], r["col_ptr"]) and np.array_equal(g["in_edge"], r["in_edge"])
    check_edge_invariants(g["src"], g["dst"], g["row_ptr"], b.plane, b.event_offsets, cfg.k, cfg.window)


@pytest.mark.parametrize("k,w,d2max", [(4, 1, np.inf), (10, 2, np.inf), (16, 3, 2.0), (3, 25, np.inf), (33, 2, np.inf),
                                       (50, 2, 1.0), (50, 2, 9.0), (64, 3, 1e30), (10, 2, 3.0), (7, 1, 1e-3)])
def test_knn_ties_duplicates_radius_and_ragged_events(k, w, d2max):
    # integer-valued embeddings: many exact ties and duplicated points; events of ragged sizes incl. empty
    rng = np.random.default_rng(100 + k)
    sizes = [0, 37, 1, 0, 900, 130, 0]
    planes, off = [], [0]
    for n in sizes:
        planes.append(np.sort(rng.integers(0, 26, n)).astype(np.int32)); off.append(off[-1] + n)
    plane = np.concatenate(planes); off = np.asarray(off, np.int32)
    emb = np.round(rng.normal(0, 1.5, (plane.size, 4))).astype(F)
    cfg = datagen.get_config("cfg1").replace(k=k, window=w, d2_max=float(d2max), precision="fp32", gnn_iters=1)
    blob = datagen.pack_blob(cfg, datagen.make_weights(cfg, "parity"))
    b = datagen.EventBatch(np.zeros((plane.size, 3), F), plane, off, np.zeros(plane.size, np.int64))
    nbr, deg = oracle.knn(emb, plane, off, k, w, d2max)
    src, dst, row_ptr = oracle.build_edges(nbr, deg)
    col_ptr, in_edge = oracle.csc(dst, plane.size)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, emb=emb, last_stage=3)
    assert np.array_equal(g["src"], src) and np.array_equal(g["dst"], dst)
    assert np.array_equal(g["row_ptr"], row_ptr) and np.array_equal(g["col_ptr"], col_ptr)
    assert np.array_equal(g["in_edge"], in_edge)


@pytest.mark.parametrize("d2max", [0.05, 0.6, 50.0])
def test_knn_radius_cut_kernel_short_lists_overflowing_lists_and_several_tiles(d2max):
    # a finite cut takes the collect-then-sort kernel: 0.05 leaves a handful of candidates per hit (the paper's regime),
    # 0.6 puts some hits above its 64-entry list and others below (flagged buckets are redone by the insertion kernel),
    # 50.0 overflows every list; 1400 candidates per query span three of its 512-candidate tiles
    rng = np.random.default_rng(11)
    n0, n1, n2 = 300, 1400, 90
    plane = np.concatenate([np.full(n0, 4), np.full(n1, 5), np.full(n2, 6)]).astype(np.int32)
    off = np.array([0, plane.size], np.int32)
    emb = rng.normal(0, 1, (plane.size, 4)).astype(F)
    emb[:40] = np.round(emb[:40])                        # some exact ties
    emb[n0:n0 + 200] = np.round(emb[n0:n0 + 200])
    cfg = datagen.get_config("cfg5").replace(precision="fp32", gnn_iters=1, d2_max=d2max, window=1)
    blob = datagen.pack_blob(cfg, datagen.make_weights(cfg, "parity"))
    b = datagen.EventBatch(np.zeros((plane.size, 3), F), plane, off, np.zeros(plane.size, np.int64))
    nbr, deg = oracle.knn(emb, plane, off, cfg.k, cfg.window, d2max)
    inside = deg[:n0]
    if d2max == 0.05:
        assert inside.max() < 50
    if d2max == 50.0:
        assert inside.min() == 50
    src, dst, _ = oracle.build_edges(nbr, deg)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, emb=emb, last_stage=3)
    assert np.array_equal(g["src"], src) and np.array_equal(g["dst"], dst)
    ctx.destroy()


@pytest.mark.parametrize("seed", range(10))
def test_knn_seeded_random_shapes_cuts_and_k(seed):
    # random k (1..64), window, cut (none / loose / tight), bucket sizes from empty to a few hundred hits, embeddings
    # with a random share of exact duplicates: both k-NN kernels against the oracle, edge lists as arrays
    rng = np.random.default_rng(4000 + seed)
    k = int(rng.choice([1, 2, 4, 5, 10, 11, 16, 17, 32, 33, 50, 64]))
    w = int(rng.integers(1, 5))
    n_ev = int(rng.integers(1, 5))
    planes, off = [], [0]
    for _ in range(n_ev):
        per_plane = rng.integers(0, int(rng.choice([3, 40, 300])), 26)
        per_plane[rng.random(26) < 0.2] = 0
        planes.append(np.repeat(np.arange(26), per_plane).astype(np.int32)); off.append(off[-1] + int(per_plane.sum()))
    plane = np.concatenate(planes); off = np.asarray(off, np.int32)
    emb = rng.normal(0, 1, (plane.size, 4)).astype(F)
    dup = rng.random(plane.size) < rng.choice([0.0, 0.3, 0.9])
    emb[dup] = np.round(emb[dup])
    d2max = float(rng.choice([np.inf, 30.0, 1.5, 0.2, 1e-4]))
    cfg = datagen.get_config("cfg1").replace(k=k, window=w, d2_max=d2max, precision="fp32", gnn_iters=1)
    blob = datagen.pack_blob(cfg, datagen.make_weights(cfg, "parity"))
    b = datagen.EventBatch(np.zeros((plane.size, 3), F), plane, off, np.zeros(plane.size, np.int64))
    nbr, deg = oracle.knn(emb, plane, off, k, w, d2max)
    src, dst, row_ptr = oracle.build_edges(nbr, deg)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, emb=emb, last_stage=3)
    assert np.array_equal(g["row_ptr"], row_ptr), (k, w, d2max)
    assert np.array_equal(g["src"], src) and np.array_equal(g["dst"], dst), (k, w, d2max)
    ctx.destroy()


def test_knn_candidate_window_larger_than_the_shared_memory_tile():
    # one event, two planes, 3000 candidates per query: spans several 1024-candidate tiles + a ragged tail
    rng = np.random.default_rng(7)
    n0, n1 = 150, 3000
    plane = np.concatenate([np.full(n0, 10), np.full(n1, 11)]).astype(np.int32)
    off = np.array([0, n0 + n1], np.int32)
    emb = rng.normal(0, 1, (n0 + n1, 4)).astype(F)
    cfg = datagen.get_config("cfg4").replace(precision="fp32", gnn_iters=1)
    blob = datagen.pack_blob(cfg, datagen.make_weights(cfg, "parity"))
    b = datagen.EventBatch(np.zeros((plane.size, 3), F), plane, off, np.zeros(plane.size, np.int64))
    nbr, deg = oracle.knn(emb, plane, off, cfg.k, cfg.window)
    src, dst, _ = oracle.build_edges(nbr, deg)
    g = run_gpu(make_ctx(cfg, blob, b), b, emb=emb, last_stage=3)
    assert np.array_equal(g["src"], src) and np.array_equal(g["dst"], dst)


# ---------------------------------------------------------------------------------- S1
@pytest.mark.parametrize("name,precision", [("cfg0", "fp32"), ("cfg1", "fp32"), ("cfg1", "bf16"), ("cfg1", "int8")])
def test_embedding_simt_engine_bit_exact(name, precision):
    cfg, b, W = _setup(name, 3 if name != "cfg0" else 1, precision=precision)
    scales = None
    if precision == "int8":
        scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window)
    blob = datagen.pack_blob(cfg, W, scales)
    want = oracle.Oracle(blob, precision).embed(b.xyz)
    ctx = make_ctx(cfg, blob, b, engine="simt")
    g = run_gpu(ctx, b, last_stage=1)
    assert np.array_equal(g["emb"], want)


# ---------------------------------------------------------------------------------- S4
@pytest.mark.parametrize("name,n_events,eei", [("cfg0", 1, 0), ("cfg1", 3, 0), ("cfg0", 1, 1)])
def test_gnn_fp32_on_oracle_edges(name, n_events, eei):
    cfg, b, W = _setup(name, n_events, precision="fp32")
    if eei:
        cfg = cfg.replace(edge_enc_input=1)
        W = datagen.make_weights(cfg, "parity")
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "fp32")
    og = o.gnn(b.xyz, r["src"], r["dst"], want_states=True, m_iter=cfg.gnn_iters - 1)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, emb=r["emb"], src=r["src"], dst=r["dst"], last_stage=5)
    d = cfg.gnn_latent
    assert np.array_equal(state(ctx, "m", b.n_hits, 2 * d), og["m"])          # ascending-edge-id sums (R22)
    assert np.array_equal(state(ctx, "h", b.n_hits, d), og["h"])
    assert np.array_equal(state(ctx, "e", r["src"].size, d), og["e"])
    assert np.array_equal(g["logit"], og["logit"])                            # pinned order => bit-exact
    assert np.abs(g["score"] - og["score"]).max() <= 1e-4                     # north_star fp32 bar
    assert np.array_equal(g["track_id"], r["track_id"])
    mid = np.mean((og["score"] > 0.01) & (og["score"] < 0.99))
    assert mid > 0.5, "scores must be informative for this comparison to mean anything"


@pytest.mark.parametrize("precision", ["bf16", "int8"])
def test_gnn_simt_engine_reproduces_the_oracles_rounding_points(precision):
    cfg, b, W = _setup("cfg1", 2, precision=precision)
    scales = None
    if precision == "int8":
        scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window)
    blob = datagen.pack_blob(cfg, W, scales)
    o, r = _oracle_all(cfg, b, blob, precision)
    og = o.gnn(b.xyz, r["src"], r["dst"], want_states=True)
    ctx = make_ctx(cfg, blob, b, engine="simt")
    g = run_gpu(ctx, b, emb=r["emb"], src=r["src"], dst=r["dst"])
    assert np.array_equal(state(ctx, "e", r["src"].size, cfg.gnn_latent), og["e"])
    assert np.array_equal(g["logit"], og["logit"])
    assert np.abs(g["score"] - og["score"]).max() <= (2e-2 if precision == "bf16" else 1e-4)


def test_int8_accumulators_bit_exact_simt_engine():
    cfg, b, W = _setup("cfg1", 2, precision="int8")
    scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window)
    blob = datagen.pack_blob(cfg, W, scales)
    o, r = _oracle_all(cfg, b, blob, "int8")
    names = [n for n, _, _ in datagen.layer_shapes(cfg)]
    ctx = make_ctx(cfg, blob, b, engine="simt")
    for lname, rows in (("emb2", b.n_hits), ("node3_0", b.n_hits), ("edge5_0", r["src"].size), ("edge0_1", r["src"].size)):
        li = names.index(lname)
        width = datagen.layer_shapes(cfg)[li][1]
        tap = np.zeros((rows, width), np.int32)
        o.set_tap(li, tap)
        o.embed(b.xyz); o.gnn(b.xyz, r["src"], r["dst"])
        o.set_tap(-1, None)
        ctx.tap_layer(li)
        run_gpu(ctx, b, emb=r["emb"] if not lname.startswith("emb") else None, src=r["src"], dst=r["dst"])
        got = ctx.buffer("tap", torch.int32).cpu().numpy()[: rows * width].reshape(rows, width)
        ctx.tap_layer(-1)
        assert np.array_equal(got, tap), lname
        assert np.abs(tap).max() > 100


# ---------------------------------------------------------------------------------- S5
def test_components_bit_exact_on_oracle_logits():
    cfg, b, W = _setup("cfg1", 6, precision="fp32")
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "fp32")
    ctx = make_ctx(cfg, blob, b)
    rng = np.random.default_rng(3)
    for trial, logit in enumerate([r["logit"], rng.normal(0, 1, r["src"].size).astype(F),
                                   rng.normal(2.5, 1, r["src"].size).astype(F), np.full(r["src"].size, -1, F),
                                   np.zeros(r["src"].size, F)]):
        want = oracle.components(r["src"], r["dst"], logit, oracle.logit_threshold(cfg.threshold), b.n_hits)
        g = run_gpu(ctx, b, emb=r["emb"], src=r["src"], dst=r["dst"], logit=logit)
        assert np.array_equal(g["track_id"], want), trial
        check_track_invariants(g["track_id"], r["src"], r["dst"], logit >= 0, b.event_offsets)


# ---------------------------------------------------------------------------------- end to end
@pytest.mark.parametrize("name,n_events,preset", [("cfg0", 1, "parity"), ("cfg0", 1, "he"), ("cfg1", 6, "parity"),
                                                   ("cfg1", 3, "he")])
def test_end_to_end_fp32_bit_exact_edges_and_track_ids(name, n_events, preset):
    cfg, b, W = _setup(name, n_events, preset=preset, precision="fp32")
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "fp32")
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)                     # the plain etx_run call
    assert np.array_equal(g["emb"], r["emb"])
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"])
    assert np.abs(g["score"] - r["score"]).max() <= 1e-4
    assert np.array_equal(g["track_id"], r["track_id"])
    assert np.unique(g["track_id"]).size == np.unique(r["track_id"]).size


@pytest.mark.parametrize("name,n_events,precision", [("cfg0", 1, "fp32"), ("cfg1", 4, "fp32"), ("cfg1", 4, "bf16"),
                                                      ("cfg5", 3, "bf16")])
def test_cylindrical_embedding_input(name, n_events, precision):
    # L96 / R27: the embedding reads normalised (r, phi, z).  Every step of R27 is a single pinned fp32 operation, so
    # the features equal the oracle's bits in every precision; fp32 then stays bit-exact end to end
    cfg = datagen.get_config(name).replace(emb_input=1, precision=precision)
    b = datagen.generate_batch(cfg, n_events=n_events)
    xyz = b.xyz.copy()
    xyz[0, :2] = (0.0, 0.0); xyz[1, :2] = (-7.0, 0.0); xyz[2, :2] = (0.0, -9.0); xyz[3, :2] = (-6.0, -6.0)   # axes, diagonal
    xyz[4, :2] = (-0.0, 5.0); xyz[5, :2] = (-8.0, -0.0)
    b = datagen.EventBatch(xyz, b.plane, b.event_offsets, b.particle)
    W = centred_parity_weights(cfg, b)
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, precision)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    fe = ctx.buffer("feat_emb", torch.float32).cpu().numpy().reshape(-1, 4)[:b.n_hits]
    fc = ctx.buffer("feat", torch.float32).cpu().numpy().reshape(-1, 4)[:b.n_hits]
    assert np.array_equal(fe[:, :3], o.features_emb(b.xyz)) and np.array_equal(fc[:, :3], o.features(b.xyz))
    assert not np.array_equal(fe, fc)
    if precision == "fp32":
        assert np.array_equal(g["emb"], r["emb"])
        assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"])
        assert np.abs(g["score"] - r["score"]).max() <= 1e-4
        assert np.array_equal(g["track_id"], r["track_id"])
    else:
        assert np.abs(g["emb"] - r["emb"]).max() <= 2e-2 * max(1.0, float(np.abs(r["emb"]).max()))
        nbr, deg = oracle.knn(g["emb"], b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max)   # chained (sec. 6)
        src, dst, _ = oracle.build_edges(nbr, deg)
        assert np.array_equal(g["src"], src) and np.array_equal(g["dst"], dst)
        og = o.gnn(b.xyz, src, dst)
        assert np.abs(g["score"] - og["score"]).max(initial=0.0) <= 2e-2
        tid = oracle.components(src, dst, g["logit"], oracle.logit_threshold(cfg.threshold), b.n_hits)
        assert np.array_equal(g["track_id"], tid)
    # a blob that says Cartesian is refused by a handle that says cylindrical
    with pytest.raises(Exception):
        make_ctx(cfg, datagen.pack_blob(cfg.replace(emb_input=0), W), b)
    ctx.destroy()


def test_one_huge_event_takes_the_global_memory_paths():
    # maximum sizes: twenty events merged into one of ~42,000 hits with ~1,600 hits per plane -- more than the 16,384
    # hits the per-event union-find keeps in shared memory and more than the 1,024 cursors per bucket of the CSC walk, so
    # both kernels run on their global-memory scratch; the k-NN walks several candidate tiles per bucket.  fp32: bit-exact
    cfg = datagen.get_config("cfg1")
    b20 = datagen.generate_batch(cfg, n_events=20)
    order = np.argsort(b20.plane, kind="stable")
    big = datagen.EventBatch(b20.xyz[order], b20.plane[order], np.array([0, b20.n_hits], np.int32), b20.particle[order])
    small = datagen.generate_batch(cfg, n_events=2, seed=77)
    b = datagen.EventBatch(np.concatenate([small.xyz, big.xyz]), np.concatenate([small.plane, big.plane]),
                           np.concatenate([small.event_offsets, [small.n_hits + big.n_hits]]).astype(np.int32),
                           np.concatenate([small.particle, big.particle]))
    assert big.n_hits > 16384 and np.bincount(big.plane).max() > 1024
    W = centred_parity_weights(cfg, small)
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "fp32")
    ctx = make_ctx(cfg, blob, b, validate=True)
    g = run_gpu(ctx, b)
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"])
    assert np.array_equal(g["col_ptr"], r["col_ptr"]) and np.array_equal(g["in_edge"], r["in_edge"])
    assert np.abs(g["score"] - r["score"]).max() <= 1e-4
    assert np.array_equal(g["track_id"], r["track_id"])
    t = ctx.tracks(b.n_hits, b.n_events, 3)
    want = oracle.tracks(r["track_id"], b.event_offsets, 3)
    for key in ("track_index", "track_offsets", "track_hits", "event_track_offsets"):
        assert np.array_equal(t[key].cpu().numpy(), want[key]), key
    ctx.destroy()


@pytest.mark.parametrize("name,precision", [("cfg1", "bf16"), ("cfg5", "bf16"), ("cfg1", "int8")])
def test_plain_run_skips_the_dead_final_edge_state_and_changes_nothing_else(name, precision):
    # e^L feeds only the classifier (L142), which is fused into the last edge network: etx_run does not write it back,
    # etx_dbg_run does.  Logits, scores and track ids must be the same bits either way
    cfg, b, W = _setup(name, 3, precision=precision)
    blob = _int8_blob(cfg, b, W) if precision == "int8" else datagen.pack_blob(cfg, W)
    ctx = make_ctx(cfg, blob, b)
    g1 = run_gpu(ctx, b, debug=False)
    e1 = state(ctx, "e", g1["n_edges"], cfg.gnn_latent).copy()
    g2 = run_gpu(ctx, b)
    e2 = state(ctx, "e", g2["n_edges"], cfg.gnn_latent)
    for key in ("src", "logit", "score", "track_id"):
        assert np.array_equal(g1[key], g2[key]), key
    assert not np.array_equal(e1, e2)                    # the plain run left e^(L-1) in place
    ctx.destroy()


@pytest.mark.parametrize("d,eei,precision", [(32, 1, "bf16"), (64, 1, "bf16"), (64, 0, "bf16"), (32, 0, "bf16"),
                                             (64, 0, "fp32"), (64, 1, "int8"), (64, 0, "int8")])
def test_no_message_passing_steps_classifier_on_the_encoded_edges(d, eei, precision):
    # degenerate case L = 0: the classifier reads e0 straight from the edge encoder (the head is fused into the encoder
    # launch); with the paper's encoder input (L133) that is the edge-network kernel in its no-old-state mode
    cfg = datagen.get_config("cfg1").replace(precision=precision, gnn_latent=d, gnn_iters=0, edge_enc_input=eei)
    b = datagen.generate_batch(cfg, n_events=3)
    W = centred_parity_weights(cfg.replace(precision="fp32") if precision == "int8" else cfg, b)
    blob = _int8_blob(cfg, b, W) if precision == "int8" else datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, precision)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, emb=r["emb"], src=r["src"], dst=r["dst"])
    og = o.gnn(b.xyz, r["src"], r["dst"], want_states=True)
    tol = 2e-2 if precision == "bf16" else 1e-4
    assert np.abs(g["score"] - og["score"]).max() <= tol
    assert np.mean((og["score"] > 0.01) & (og["score"] < 0.99)) > 0.3          # the comparison is informative
    e = state(ctx, "e", r["src"].size, d)
    assert np.abs(e - og["e"]).max() <= tol * max(1.0, float(np.abs(og["e"]).max()))
    if precision == "int8":
        assert np.array_equal(g["logit"], og["logit"])
    g2 = run_gpu(ctx, b, debug=False)
    assert np.array_equal(g2["track_id"], oracle.components(g2["src"], g2["dst"], g2["logit"], oracle.logit_threshold(cfg.threshold), b.n_hits))
    ctx.destroy()


@pytest.mark.parametrize("thr", [0.0, 1.0, 0.999, 1e-3])
def test_threshold_extremes(thr):
    # s_edge,min = 0 keeps every edge (components = those of the rough graph), 1 keeps none unless a score is exactly 1
    # (every hit its own track on these weights); the decision is taken on the logit (R17)
    cfg, b, W = _setup("cfg1", 3, precision="fp32")
    cfg = cfg.replace(threshold=thr)
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "fp32")
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["track_id"], r["track_id"])
    n_tracks = np.unique(g["track_id"]).size
    if thr == 0.0:
        import scipy.sparse as sp
        from scipy.sparse.csgraph import connected_components
        A = sp.coo_matrix((np.ones(r["src"].size), (r["src"], r["dst"])), shape=(b.n_hits, b.n_hits))
        assert n_tracks == connected_components(A, directed=False)[0]
    if thr == 1.0:
        assert n_tracks == b.n_hits
    ctx.destroy()


def test_repeated_runs_on_one_handle_are_identical_and_smaller_batches_work():
    cfg, b, W = _setup("cfg1", 4, precision="fp32")
    blob = datagen.pack_blob(cfg, W)
    ctx = make_ctx(cfg, blob, b)
    g1 = run_gpu(ctx, b, debug=False)
    b2 = b.slice_events(1, 3)
    g2 = run_gpu(ctx, b2, debug=False)
    r2 = oracle.Oracle(blob, "fp32").run(b2.xyz, b2.plane, b2.event_offsets, cfg.k, cfg.window)
    assert np.array_equal(g2["src"], r2["src"]) and np.array_equal(g2["track_id"], r2["track_id"])
    g3 = run_gpu(ctx, b, debug=False)
    for key in ("src", "dst", "logit", "track_id"):
        assert np.array_equal(g1[key], g3[key])


# ---------------------------------------------------------------------------------- edge cases + errors
def test_empty_batches_and_empty_events():
    cfg = datagen.get_config("cfg0")
    W = datagen.make_weights(cfg, "parity")
    blob = datagen.pack_blob(cfg, W)
    empty = datagen.EventBatch(np.zeros((0, 3), F), np.zeros(0, np.int32), np.zeros(1, np.int32), np.zeros(0, np.int64))
    ctx = make_ctx(cfg, blob, empty, max_events=8, max_hits=4096)
    g = run_gpu(ctx, empty, debug=False)                                   # n_events = 0
    assert g["n_edges"] == 0 and g["track_id"].size == 0
    empty3 = datagen.EventBatch(np.zeros((0, 3), F), np.zeros(0, np.int32), np.zeros(4, np.int32), np.zeros(0, np.int64))
    g = run_gpu(ctx, empty3, debug=False)                                  # three empty events
    assert g["n_edges"] == 0
    b = datagen.generate_batch(cfg, n_events=2)
    o = b.event_offsets
    off = np.array([0, 0, o[1], o[1], o[1], o[2], o[2]], np.int32)         # empty first / middle / last events
    bb = datagen.EventBatch(b.xyz, b.plane, off, b.particle)
    r = oracle.Oracle(blob, "fp32").run(bb.xyz, bb.plane, bb.event_offsets, cfg.k, cfg.window)
    g = run_gpu(ctx, bb, debug=False)
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["track_id"], r["track_id"])
    # a hit on plane 25 only, and a single-hit event
    hb = datagen.hand_batch([[(10.0, 0.0, 25)], [(7.0, 7.0, 3)], [(10.0, 1.0, 3), (10.1, 1.0, 4), (10.2, 1.1, 5)]])
    r = oracle.Oracle(blob, "fp32").run(hb.xyz, hb.plane, hb.event_offsets, cfg.k, cfg.window)
    g = run_gpu(ctx, hb, debug=False)
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"])
    assert np.array_equal(g["track_id"], r["track_id"]) and g["n_edges"] == 2


def test_error_codes_capacity_blob_order_unsupported():
    import paper_2407_12119_b200 as etx
    cfg = datagen.get_config("cfg0")
    W = datagen.make_weights(cfg, "parity")
    blob = datagen.pack_blob(cfg, W)
    b = datagen.generate_batch(cfg, n_events=2)
    with pytest.raises(etx.EtxError) as ei:
        make_ctx(cfg, blob[:-4], b)
    assert ei.value.status == -2
    with pytest.raises(etx.EtxError) as ei:
        make_ctx(cfg, b"\0" * len(blob), b)
    assert ei.value.status == -2
    with pytest.raises(etx.EtxError) as ei:
        make_ctx(cfg.replace(gnn_latent=48), datagen.pack_blob(cfg.replace(gnn_latent=48), datagen.make_weights(cfg.replace(gnn_latent=48))), b)
    assert ei.value.status == -6
    # state_dtype: bf16 state needs bf16 or int8 precision, fp32 state fp32 or int8 (include/etx.h)
    for prec, st in (("fp32", "bf16"), ("bf16", "fp32")):
        with pytest.raises(etx.EtxError) as ei:
            make_ctx(cfg.replace(precision=prec, state_dtype=st), blob, b)
        assert ei.value.status == -6
    ctx = make_ctx(cfg, blob, b, max_events=1, max_hits=b.n_hits, validate=True)
    with pytest.raises(etx.EtxError) as ei:
        run_gpu(ctx, b, debug=False)
    assert ei.value.status == -3
    ctx = make_ctx(cfg, blob, b, max_events=4, max_hits=10)
    with pytest.raises(etx.EtxError) as ei:
        run_gpu(ctx, b, debug=False)
    assert ei.value.status == -3
    # unsorted planes are detected on the device; the batch is rejected THERE (no edges, every hit its own track),
    # the verdict is read after synchronising, and the next (valid) batch runs normally
    ctx = make_ctx(cfg, blob, b, validate=True)
    bad = datagen.EventBatch(b.xyz, b.plane[::-1].copy(), b.event_offsets, b.particle)
    r = ctx.results(ctx.run(dev(bad.xyz), dev(bad.plane), bad.event_offsets))
    torch.cuda.synchronize()
    assert ctx.input_status() == -4
    assert r["n_edges"] == 0 and np.array_equal(r["track_id"].cpu().numpy(), np.arange(b.n_hits, dtype=np.int32))
    oob = b.plane.copy(); oob[3] = 26                                      # a plane index out of range
    ctx.results(ctx.run(dev(b.xyz), dev(oob), b.event_offsets))
    torch.cuda.synchronize()
    assert ctx.input_status() == -4
    # etx_run_host synchronises and reports the same batch
    cap = cfg.k * b.n_hits
    hs = torch.empty(cap, dtype=torch.float32).pin_memory(); hi = torch.empty(cap, dtype=torch.int32).pin_memory()
    hj = torch.empty(cap, dtype=torch.int32).pin_memory(); ht = torch.empty(b.n_hits, dtype=torch.int32).pin_memory()
    with pytest.raises(etx.EtxError) as ei:
        ctx.run_host(torch.from_numpy(bad.xyz).pin_memory(), torch.from_numpy(bad.plane).pin_memory(), bad.event_offsets, hs, hi, hj, ht)
    assert ei.value.status == -4
    E = ctx.run_host(torch.from_numpy(b.xyz).pin_memory(), torch.from_numpy(b.plane).pin_memory(), b.event_offsets, hs, hi, hj, ht)
    assert E > 0 and ctx.input_status() == 0
    g = run_gpu(ctx, b, debug=False)                                       # the handle stays usable
    assert g["n_edges"] > 0


@pytest.mark.parametrize("precision,pinned", [("fp32", True), ("fp32", False), ("bf16", True), ("bf16", False)])
def test_run_host_matches_device_run(precision, pinned):
    # pinned buffers: src / dst are copied under the GNN and the scores are written by the classifier straight into
    # the (device-addressable) host buffer; pageable buffers: plain copies after the run.  Same bits either way.
    cfg, b, W = _setup("cfg1", 3, precision=precision)
    blob = datagen.pack_blob(cfg, W)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    cap = cfg.k * b.n_hits
    mk = (lambda t: t.pin_memory()) if pinned else (lambda t: t)
    h_xyz = mk(torch.from_numpy(b.xyz)); h_plane = mk(torch.from_numpy(b.plane))
    sc = mk(torch.full((cap,), -1.0, dtype=torch.float32)); s_ = mk(torch.empty(cap, dtype=torch.int32))
    d_ = mk(torch.empty(cap, dtype=torch.int32)); tid = mk(torch.empty(b.n_hits, dtype=torch.int32))
    for _ in range(2):                                       # twice: the direct-write redirection must not stick
        E = ctx.run_host(h_xyz, h_plane, b.event_offsets, sc, s_, d_, tid)
        assert E == g["n_edges"]
        assert np.array_equal(s_.numpy()[:E], g["src"]) and np.array_equal(d_.numpy()[:E], g["dst"])
        assert np.array_equal(sc.numpy()[:E], g["score"]) and np.array_equal(tid.numpy(), g["track_id"])
        assert (sc.numpy()[E:] == -1.0).all()                # nothing is written behind the E scores
    g2 = run_gpu(ctx, b, debug=False)                        # and a device run afterwards still fills its own buffer
    assert np.array_equal(g2["score"], g["score"])


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_submit_host_pipelined_matches_run_host(precision):
    import paper_2407_12119_b200 as etx
    # etx_submit_host / etx_wait_host: two submissions in flight, inputs copied under the previous batch's compute, the
    # edge list written to the host by the device itself.  Different batches alternate, so any cross-talk between the
    # two staging sets or output buffers would show.
    cfg, b, W = _setup("cfg1", 4, precision=precision)
    blob = datagen.pack_blob(cfg, W)
    batches = [b.slice_events(0, 2), b.slice_events(1, 4), b.slice_events(2, 3), b, b.slice_events(0, 1)]
    ctx = make_ctx(cfg, blob, b, validate=True)
    want = [run_gpu(ctx, x, debug=False) for x in batches]
    cap = cfg.k * b.n_hits
    pin = lambda *shape, dtype: torch.empty(*shape, dtype=dtype).pin_memory()
    bufs = [dict(sc=pin(cap, dtype=torch.float32), s=pin(cap, dtype=torch.int32), d=pin(cap, dtype=torch.int32),
                 t=pin(b.n_hits, dtype=torch.int32), n=torch.zeros(1, dtype=torch.int32)) for _ in range(2)]
    hx = [torch.from_numpy(x.xyz).pin_memory() for x in batches]; hp = [torch.from_numpy(x.plane).pin_memory() for x in batches]
    tickets = []

    def check(i):
        ctx.wait_host(tickets[i])
        o, w = bufs[i & 1], want[i]
        E = int(o["n"][0])
        assert E == w["n_edges"], i
        assert np.array_equal(o["s"].numpy()[:E], w["src"]) and np.array_equal(o["d"].numpy()[:E], w["dst"]), i
        assert np.array_equal(o["sc"].numpy()[:E], w["score"]), i
        assert np.array_equal(o["t"].numpy()[:batches[i].n_hits], w["track_id"]), i

    for rep in range(2):
        tickets.clear()
        for i, x in enumerate(batches):
            o = bufs[i & 1]
            tickets.append(ctx.submit_host(hx[i], hp[i], x.event_offsets, o["sc"], o["s"], o["d"], o["t"], o["n"]))
            if i >= 1:
                check(i - 1)
        check(len(batches) - 1)
    # pageable output buffers are refused (the device writes them itself); a rejected batch reports on ITS ticket
    with pytest.raises(etx.EtxError) as ei:
        ctx.submit_host(hx[0], hp[0], batches[0].event_offsets, torch.empty(cap), bufs[0]["s"], bufs[0]["d"], bufs[0]["t"], bufs[0]["n"])
    assert ei.value.status == -1
    bad = torch.from_numpy(batches[0].plane[::-1].copy()).pin_memory()
    t_bad = ctx.submit_host(hx[0], bad, batches[0].event_offsets, bufs[0]["sc"], bufs[0]["s"], bufs[0]["d"], bufs[0]["t"], bufs[0]["n"])
    t_ok = ctx.submit_host(hx[1], hp[1], batches[1].event_offsets, bufs[1]["sc"], bufs[1]["s"], bufs[1]["d"], bufs[1]["t"], bufs[1]["n"])
    with pytest.raises(etx.EtxError) as ei:
        ctx.wait_host(t_bad)
    assert ei.value.status == -4 and int(bufs[0]["n"][0]) == 0
    # other calls on the handle are refused while a submission is outstanding, and work again afterwards
    with pytest.raises(etx.EtxError) as ei:
        run_gpu(ctx, batches[0], debug=False)
    assert ei.value.status == -1
    ctx.wait_host(t_ok)
    assert int(bufs[1]["n"][0]) == want[1]["n_edges"]
    g = run_gpu(ctx, batches[0], debug=False)
    assert np.array_equal(g["score"], want[0]["score"])
    # an empty batch goes through the pipeline too
    empty = b.slice_events(0, 0)
    t = ctx.submit_host(hx[0], hp[0], np.zeros(1, np.int32), bufs[0]["sc"], bufs[0]["s"], bufs[0]["d"], bufs[0]["t"], bufs[0]["n"])
    ctx.wait_host(t)
    assert int(bufs[0]["n"][0]) == 0
    # a third submission while neither of the first two has been waited for is refused (it would reuse the first one's
    # slot: verdict, E, device score buffer); the two in flight are unharmed, and the slot is free again after its wait
    tickets.clear()
    for i in (0, 1):
        o = bufs[i]
        tickets.append(ctx.submit_host(hx[i], hp[i], batches[i].event_offsets, o["sc"], o["s"], o["d"], o["t"], o["n"]))
    with pytest.raises(etx.EtxError) as ei:
        ctx.submit_host(hx[2], hp[2], batches[2].event_offsets, bufs[0]["sc"], bufs[0]["s"], bufs[0]["d"], bufs[0]["t"], bufs[0]["n"])
    assert ei.value.status == -1
    check(0)
    tickets.append(ctx.submit_host(hx[2], hp[2], batches[2].event_offsets, bufs[0]["sc"], bufs[0]["s"], bufs[0]["d"], bufs[0]["t"], bufs[0]["n"]))
    check(1)
    check(2)
    ctx.destroy()


# ================================================================================== INT8 calibration in the product
@pytest.mark.parametrize("name,triplets", [("cfg1", 0), ("cfg0", 1), ("cfg5", 0)])
def test_calibrate_scales_equal_the_oracle_bit_for_bit(name, triplets):
    # etx_calibrate (R21): the fp32 FFMA engine is bit-exact against the oracle's fp32 forward and a
    # maximum does not depend on the order it is taken in, so the 16-event calibration batch must give the oracle's
    # activation scales to the bit -- the oracle checks the product's calibration instead of supplying it.
    import paper_2407_12119_b200 as etx
    cfg = datagen.get_config(name).replace(precision="fp32", triplets=triplets)
    cal = datagen.generate_batch(datagen.get_config("cfg1"), n_events=datagen.configs.CALIBRATION_EVENTS, seed=datagen.configs.CALIBRATION_SEED)
    W = datagen.make_weights(cfg, "parity")
    blob = datagen.pack_blob(cfg, W)
    want = oracle.calibrate_int8(blob, cal.xyz, cal.plane, cal.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    ctx = make_ctx(cfg, blob, cal, max_triplets=8_000_000 if triplets else 0)
    got = ctx.calibrate(dev(cal.xyz), dev(cal.plane), cal.event_offsets)
    assert got.size == want.size == datagen.weights.n_act_scales(cfg) and got.size >= 10
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32)), np.flatnonzero(got != want)
    assert (got > 0).all() and not np.all(got == 1.0)
    # a second call on the same handle starts from zero again, and an ordinary run afterwards is unaffected
    small = cal.slice_events(0, 3)
    got2 = ctx.calibrate(dev(small.xyz), dev(small.plane), small.event_offsets)
    want2 = oracle.calibrate_int8(blob, small.xyz, small.plane, small.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    assert np.array_equal(got2.view(np.uint32), want2.view(np.uint32)) and (got2 <= got).all()
    g = run_gpu(ctx, small, debug=False)
    assert g["n_edges"] > 0
    ctx.destroy()
    # the scales make a valid INT8 blob; a bf16 handle cannot calibrate
    cfg8 = cfg.replace(precision="int8")
    ctx8 = make_ctx(cfg8, datagen.pack_blob(cfg8, W, got), small, max_triplets=8_000_000 if triplets else 0)
    assert run_gpu(ctx8, small, debug=False)["n_edges"] > 0      # (with a radius cut the quantised embedding moves a few edges)
    with pytest.raises(etx.EtxError) as ei:
        ctx8.calibrate(dev(small.xyz), dev(small.plane), small.event_offsets)
    assert ei.value.status == -6
    ctx8.destroy()


# ================================================================================== tcgen05 engine (bf16 / int8)
def _int8_blob(cfg, b, W):
    scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window)
    return datagen.pack_blob(cfg, W, scales)


@pytest.mark.parametrize("name,n_events", [("cfg1", 3), ("cfg0", 1)])
def test_int8_tensor_core_path_is_bit_exact_end_to_end(name, n_events):
    # integer accumulation is order-free and every non-integer op is a single pinned fp32 op (R21): the
    # tcgen05 kind::i8 path must reproduce the oracle bit for bit -- embedding, edges, logits, track ids
    cfg, b, W = _setup(name, n_events, precision="int8")
    blob = _int8_blob(cfg, b, W)
    o, r = _oracle_all(cfg, b, blob, "int8")
    og = o.gnn(b.xyz, r["src"], r["dst"], want_states=True)
    ctx = make_ctx(cfg, blob, b)                                   # engine auto -> tcgen05
    g = run_gpu(ctx, b, debug=False)
    assert np.array_equal(g["emb"], r["emb"])
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"])
    assert np.array_equal(state(ctx, "h", b.n_hits, cfg.gnn_latent), og["h"])
    assert np.array_equal(g["logit"], r["logit"])
    assert np.abs(g["score"] - r["score"]).max() <= 1e-4
    assert np.array_equal(g["track_id"], r["track_id"])
    # a plain etx_run does not write e^L back (only the fused classifier reads it); etx_dbg_run does, with the same logits
    g2 = run_gpu(ctx, b)
    assert np.array_equal(state(ctx, "e", r["src"].size, cfg.gnn_latent), og["e"])
    assert np.array_equal(g2["logit"], g["logit"]) and np.array_equal(g2["track_id"], g["track_id"])


@pytest.mark.parametrize("name,n_events,engine", [("cfg1", 3, "auto"), ("cfg0", 1, "auto"), ("cfg1", 2, "simt"), ("cfg1", 2, "tc_serial"),
                                                  ("cfg5", 1, "auto")])
def test_int8_with_bf16_state_is_bit_exact_end_to_end(name, n_events, engine):
    # state_dtype = bf16 in INT8 mode (R21 / SURVEY A21): h, e, m are stored as bf16 (RNE), every arithmetic step is
    # still the pinned fp32 / integer one, so all three engines must reproduce the oracle bit for bit
    cfg, b, W = _setup(name, n_events, precision="int8")
    cfg = cfg.replace(state_dtype="bf16")
    scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max)
    blob = datagen.pack_blob(cfg, W, scales)
    o, r = _oracle_all(cfg, b, blob, "int8")
    og = o.gnn(b.xyz, r["src"], r["dst"], want_states=True)
    ctx = make_ctx(cfg, blob, b, engine=engine)
    g = run_gpu(ctx, b, debug=False)
    assert np.array_equal(g["emb"], r["emb"])
    assert np.array_equal(g["src"], r["src"]) and np.array_equal(g["dst"], r["dst"])
    assert np.array_equal(state(ctx, "h", b.n_hits, cfg.gnn_latent), og["h"])
    assert np.array_equal(g["logit"], r["logit"])
    assert np.array_equal(g["track_id"], r["track_id"])
    g2 = run_gpu(ctx, b)                                           # etx_dbg_run writes e^L back
    assert np.array_equal(state(ctx, "e", r["src"].size, cfg.gnn_latent), og["e"])
    assert np.array_equal(state(ctx, "m", b.n_hits, 2 * cfg.gnn_latent),
                          o.gnn(b.xyz, r["src"], r["dst"], m_iter=cfg.gnn_iters - 1)["m"])
    assert np.array_equal(g2["logit"], g["logit"])
    # the stored state really is bf16, and it differs from the fp32-state result
    e = state(ctx, "e", r["src"].size, cfg.gnn_latent)
    assert np.array_equal(e, torch.from_numpy(e).to(torch.bfloat16).float().numpy())
    r32 = oracle.Oracle(blob, "int8").run(b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    assert not np.array_equal(r32["logit"], r["logit"])
    # int32 accumulators of the production kernels (AUTO engine) with the bf16 state
    if engine == "auto" and name == "cfg1":
        names = [n for n, _, _ in datagen.layer_shapes(cfg)]
        for lname, rows in (("node1_0", b.n_hits), ("edge2_0", r["src"].size), ("edge5_1", r["src"].size), ("eenc1", r["src"].size)):
            li = names.index(lname)
            tap = np.zeros((rows, cfg.gnn_latent), np.int32)
            o.set_tap(li, tap); o.gnn(b.xyz, r["src"], r["dst"]); o.set_tap(-1, None)
            ctx.tap_layer(li)
            run_gpu(ctx, b, debug=False)
            got = ctx.buffer("tap", torch.int32).cpu().numpy()[: rows * cfg.gnn_latent].reshape(rows, cfg.gnn_latent)
            ctx.tap_layer(-1)
            assert np.array_equal(got, tap), lname


def test_int8_tensor_core_accumulators_bit_exact():
    cfg, b, W = _setup("cfg1", 2, precision="int8")
    blob = _int8_blob(cfg, b, W)
    o, r = _oracle_all(cfg, b, blob, "int8")
    names = [n for n, _, _ in datagen.layer_shapes(cfg)]
    ctx = make_ctx(cfg, blob, b)
    for lname, rows in (("emb1", b.n_hits), ("emb3", b.n_hits), ("nenc1", b.n_hits), ("eenc1", r["src"].size),
                        ("node2_0", b.n_hits), ("node5_1", b.n_hits), ("edge0_0", r["src"].size), ("edge5_1", r["src"].size)):
        li = names.index(lname)
        width = datagen.layer_shapes(cfg)[li][1]
        tap = np.zeros((rows, width), np.int32)
        o.set_tap(li, tap)
        o.embed(b.xyz); o.gnn(b.xyz, r["src"], r["dst"])
        o.set_tap(-1, None)
        ctx.tap_layer(li)
        run_gpu(ctx, b, debug=False)
        got = ctx.buffer("tap", torch.int32).cpu().numpy()[: rows * width].reshape(rows, width)
        ctx.tap_layer(-1)
        assert np.array_equal(got, tap), lname
        assert np.abs(tap).max() > 100


@pytest.mark.parametrize("name,n_events", [("cfg1", 3), ("cfg0", 1), ("cfg4", 1)])
def test_bf16_tensor_core_path_stage_isolated_and_chained(name, n_events):
    cfg, b, W = _setup(name, n_events, precision="bf16")
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "bf16")
    ctx = make_ctx(cfg, blob, b)
    # S1 stage-isolated: bf16 products are exact, only the fp32 accumulation order differs from the oracle
    g1 = run_gpu(ctx, b, last_stage=1)
    assert np.abs(g1["emb"] - r["emb"]).max() <= 2e-2 * max(1.0, np.abs(r["emb"]).max())
    # S4 stage-isolated on the oracle's edge list: north_star bar 2e-2 absolute on scores
    og = o.gnn(b.xyz, r["src"], r["dst"], want_states=True)
    g = run_gpu(ctx, b, emb=r["emb"], src=r["src"], dst=r["dst"])
    err = np.abs(g["score"] - og["score"]).max()
    mid = np.mean((og["score"] > 0.01) & (og["score"] < 0.99))
    assert err <= 2e-2, err
    assert mid > 0.5
    e_gpu = state(ctx, "e", r["src"].size, cfg.gnn_latent)
    assert np.abs(e_gpu - og["e"]).max() <= 0.05 * max(1.0, np.abs(og["e"]).max())
    # chained, no injection: oracle S2 on the GPU's embedding == GPU edges; oracle S5 on GPU logits == GPU ids
    gg = run_gpu(ctx, b, debug=False)
    nbr, deg = oracle.knn(gg["emb"], b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max)
    src, dst, _ = oracle.build_edges(nbr, deg)
    assert np.array_equal(gg["src"], src) and np.array_equal(gg["dst"], dst)
    tid = oracle.components(src, dst, gg["logit"], oracle.logit_threshold(cfg.threshold), b.n_hits)
    assert np.array_equal(gg["track_id"], tid)
    og2 = o.gnn(b.xyz, src, dst)
    assert np.abs(gg["score"] - og2["score"]).max() <= 2e-2
    print(f"{name}: bf16 max|score err|={err:.2e}, edges differing from the all-oracle run: "
          f"{int(np.sum(src != r['src'][:src.size]) if src.size == r['src'].size else -1)}")


def test_bf16_tensor_core_paper_edge_encoder_and_literal_he_weights():
    cfg, b, _ = _setup("cfg1", 2, precision="bf16")
    cfg = cfg.replace(edge_enc_input=1)
    W = datagen.make_weights(cfg, "parity")
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "bf16")
    g = run_gpu(make_ctx(cfg, blob, b), b, emb=r["emb"], src=r["src"], dst=r["dst"])
    assert np.abs(g["score"] - r["score"]).max() <= 2e-2
    # literal He-uniform weights (BASELINE.json): activations blow up (R24), compare logits relatively
    cfg = datagen.get_config("cfg2")
    W = datagen.make_weights(cfg, "he")
    blob = datagen.pack_blob(cfg, W)
    o, r = _oracle_all(cfg, b, blob, "bf16")
    g = run_gpu(make_ctx(cfg, blob, b), b, emb=r["emb"], src=r["src"], dst=r["dst"])
    scale = np.abs(r["logit"]).max()
    assert np.isfinite(g["logit"]).all() and np.abs(g["logit"] - r["logit"]).max() <= 0.05 * scale


@pytest.mark.parametrize("d", [32, 64])
def test_bf16_tma_kernels_edge_cases_no_edges_tile_boundaries_and_handle_reuse(d):
    # the TMA-fed bf16 kernels (edge encoder, edge network): zero edges, one edge, edge counts on both sides of a
    # multiple of the 128-row tile, and one handle reused for a smaller batch after a larger one (stale rows behind
    # n_edges in the workspace must never leak into live rows).  Scores against the oracle on the oracle's edges.
    cfg = datagen.get_config("cfg1").replace(precision="bf16", gnn_latent=d, gnn_iters=2)
    big = datagen.generate_batch(cfg, n_events=2)
    W = centred_parity_weights(cfg, big)
    blob = datagen.pack_blob(cfg, W)
    o = oracle.Oracle(blob, "bf16")
    ctx = make_ctx(cfg, blob, big)
    r = o.run(big.xyz, big.plane, big.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    E = r["src"].size
    assert E > 1000
    for n_e in (E, 1, 127, 128, 129, 5 * 128, 5 * 128 + 1, E):       # (no edge at all: below, through S2)
        # a prefix of the oracle's (src-sorted) edge list is itself a valid src-sorted edge list
        src, dst = r["src"][:n_e], r["dst"][:n_e]
        og = o.gnn(big.xyz, src, dst)
        g = run_gpu(ctx, big, emb=r["emb"], src=src, dst=dst)
        assert g["n_edges"] == n_e
        if n_e:
            assert np.isfinite(g["score"]).all()
            assert np.abs(g["score"] - og["score"]).max() <= 2e-2, n_e
        tid = oracle.components(src, dst, g["logit"], oracle.logit_threshold(cfg.threshold), big.n_hits)
        assert np.array_equal(g["track_id"], tid), n_e
    # no candidate passes the radius cut: S2 yields no edge at all, every hit is its own track
    cfg0 = cfg.replace(d2_max=1e-30)
    ctx0 = make_ctx(cfg0, blob, big)
    g = run_gpu(ctx0, big, debug=False)
    assert g["n_edges"] == 0 and np.array_equal(g["track_id"], np.arange(big.n_hits, dtype=np.int32))


def test_two_handles_on_two_streams_run_concurrently_and_agree_with_sequential_runs():
    # One handle serves one stream at a time, several handles may run at once (include/etx.h): two bf16 handles,
    # each enqueuing several batches on its own stream without any synchronisation in between, must give the bits
    # of a sequential run (persistent one-CTA-per-SM kernels of the two streams interleave on the device).
    cfg, b, W = _setup("cfg1", 4, precision="bf16")
    blob = datagen.pack_blob(cfg, W)
    b2 = b.slice_events(1, 4)
    ref = [run_gpu(make_ctx(cfg, blob, x), x, debug=False) for x in (b, b2)]
    ctxs = [make_ctx(cfg, blob, b), make_ctx(cfg, blob, b)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ins = [(dev(x.xyz), dev(x.plane), x.event_offsets) for x in (b, b2)]
    torch.cuda.synchronize()
    outs = [None, None]
    for rep in range(3):
        for k in (0, 1):
            with torch.cuda.stream(streams[k]):
                outs[k] = ctxs[k].run(*ins[k])
    for k in (0, 1):
        with torch.cuda.stream(streams[k]):
            r = ctxs[k].results(outs[k])
        assert r["n_edges"] == ref[k]["n_edges"]
        for name in ("src", "dst", "score", "logit", "track_id"):
            assert np.array_equal(r[name].cpu().numpy(), ref[k][name]), (k, name)


def test_custom_allocator_callbacks_serve_every_device_block():
    # include/etx.h: hp.alloc / hp.dealloc (Allen-style arena).  Every device block of the handle must
    # come from the callback (sum of requests == etx_workspace_bytes), results must equal the cudaMalloc handle's,
    # every block must be handed back by etx_destroy, and a misaligned or half-specified allocator is refused.
    import ctypes as C
    import paper_2407_12119_b200 as etx
    from paper_2407_12119_b200.binding import ALLOC_FN, DEALLOC_FN
    cfg, b, W = _setup("cfg1", 2, precision="bf16")
    blob = datagen.pack_blob(cfg, W)
    ref = run_gpu(make_ctx(cfg, blob, b), b, debug=False)
    live, total = {}, [0]

    def alloc(nbytes, _ctx):
        t = torch.empty(int(nbytes) + 256, dtype=torch.uint8, device="cuda")
        p = (t.data_ptr() + 255) // 256 * 256
        live[p] = t; total[0] += int(nbytes)
        return p

    def dealloc(p, _ctx):
        if live.pop(p, None) is None:
            del live[p - 16]                                 # the deliberately misaligned block of the last case

    a_cb, d_cb = ALLOC_FN(alloc), DEALLOC_FN(dealloc)
    hp = etx.hyperparams_from_config(cfg, b.n_events, b.n_hits)
    hp.alloc, hp.dealloc = a_cb, d_cb
    ctx = etx.Etx(blob, hp)
    assert len(live) > 20 and ctx.workspace_bytes() == total[0]
    g = run_gpu(ctx, b, debug=False)
    for name in ("src", "dst", "score", "logit", "track_id"):
        assert np.array_equal(g[name], ref[name]), name
    ctx.destroy()
    assert not live
    hp2 = etx.hyperparams_from_config(cfg, b.n_events, b.n_hits)
    hp2.alloc = a_cb                                         # alloc without dealloc
    with pytest.raises(etx.EtxError):
        etx.Etx(blob, hp2)
    hp3 = etx.hyperparams_from_config(cfg, b.n_events, b.n_hits)
    hp3.alloc, hp3.dealloc = ALLOC_FN(lambda n, c: alloc(n, c) + 16), d_cb      # misaligned blocks
    with pytest.raises(etx.EtxError):
        etx.Etx(blob, hp3)


@pytest.mark.parametrize("name,n_events,precision,min_hits", [("cfg1", 5, "fp32", 3), ("cfg1", 5, "bf16", 1), ("cfg0", 1, "fp32", 3),
                                                              ("cfg4", 1, "bf16", 4)])
def test_track_containers_bit_exact_against_the_oracle(name, n_events, precision, min_hits):
    # etx_tracks regroups the run's track ids: dense numbering by smallest hit, >= min_hits filter,
    # ascending hit lists.  All integer work: every array must equal the oracle's on the GPU's own track ids.
    cfg, b, W = _setup(name, n_events, precision=precision)
    blob = datagen.pack_blob(cfg, W)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    t = ctx.tracks(b.n_hits, b.n_events, min_hits)
    r = oracle.tracks(g["track_id"], b.event_offsets, min_hits)
    assert t["n_tracks"] == r["n_tracks"] and r["n_tracks"] > 0
    for key in ("track_index", "track_offsets", "track_hits", "event_track_offsets"):
        assert np.array_equal(t[key].cpu().numpy(), r[key]), key
    # empty batch and a second call with another filter on the same handle
    t2 = ctx.tracks(b.n_hits, b.n_events, min_hits + 2)
    r2 = oracle.tracks(g["track_id"], b.event_offsets, min_hits + 2)
    assert t2["n_tracks"] == r2["n_tracks"] and np.array_equal(t2["track_hits"].cpu().numpy(), r2["track_hits"])
    ne = min(2, b.n_events)                                  # within the handle's max_events
    empty = datagen.EventBatch(np.zeros((0, 3), F), np.zeros(0, np.int32), np.zeros(ne + 1, np.int32), np.zeros(0, np.int64))
    run_gpu(ctx, empty, debug=False)
    t3 = ctx.tracks(0, ne, 3)
    assert t3["n_tracks"] == 0 and np.array_equal(t3["event_track_offsets"].cpu().numpy(), np.zeros(ne + 1, np.int32))
