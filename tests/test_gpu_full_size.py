"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (engine auto, the
whole batch in one etx_run).  The oracle cannot recompute a 500-event batch in seconds, so (DESIGN.md sec. 6,
"Full size"): properties that hold at any size are checked on the whole output, and a sample of events --
first, last, largest, smallest non-empty, a few seeded random ones -- is recomputed by the oracle one by one.
Events are independent in every stage, so an event cut out of the batch is a valid oracle
input on its own; edges and track ids are compared after rebasing hit indices."""
import numpy as np
import pytest
import torch

import datagen
import oracle
from gpu_utils import make_ctx, run_gpu
from helpers import centred_parity_weights, check_edge_invariants, check_track_invariants

pytestmark = pytest.mark.gpu


def _sample_events(b, n_random=3, seed=5):
    sizes = np.diff(b.event_offsets)
    nz = np.flatnonzero(sizes > 0)
    pick = {0, b.n_events - 1, int(np.argmax(sizes)), int(nz[np.argmin(sizes[nz])])}
    rng = np.random.default_rng(seed)
    pick.update(int(x) for x in rng.integers(0, b.n_events, n_random))
    return sorted(pick)


def _check_sampled_events(cfg, b, g, blob, precision, events, score_tol=None, logit_rel=None):
    o = oracle.Oracle(blob, precision)
    tau = oracle.logit_threshold(cfg.threshold)
    eo, rp = b.event_offsets, g["row_ptr"]
    worst = 0.0
    _, head_w, head_b = datagen.unpack_blob(cfg, blob)[0][-1]
    head_w, head_b = head_w[0], head_b[0]
    for ev in events:
        h0, h1 = int(eo[ev]), int(eo[ev + 1])
        e0, e1 = int(rp[h0]), int(rp[h1])
        sub = b.slice_events(ev, ev + 1)
        # chained: oracle S2 + S3 on the GPU's own embedding of this event == the GPU's edges (bit-exact)
        nbr, deg = oracle.knn(g["emb"][h0:h1], sub.plane, sub.event_offsets, cfg.k, cfg.window, cfg.d2_max)
        src, dst, _ = oracle.build_edges(nbr, deg)
        assert src.size == e1 - e0, (ev, src.size, e1 - e0)
        assert np.array_equal(g["src"][e0:e1] - h0, src) and np.array_equal(g["dst"][e0:e1] - h0, dst), ev
        # S4 on those edges: scores / logits within the bar
        og = o.gnn(sub.xyz, src, dst, want_states=logit_rel is not None)
        if score_tol is not None and src.size:
            err = float(np.abs(g["score"][e0:e1] - og["score"]).max())
            worst = max(worst, err)
            assert err <= score_tol, (ev, err)
        if logit_rel is not None and src.size:
            # He weights saturate every score (R24), so the logits are compared, element by element, against each
            # edge's OWN magnitude: z = w . e + b, and the bound is logit_rel * (sum_j |w_j e_ij| + |b|) -- an edge
            # with a small logit cannot hide behind the largest one of the event
            assert np.isfinite(g["logit"][e0:e1]).all()
            mag = np.abs(og["e"].astype(np.float64)) @ np.abs(head_w.astype(np.float64)) + abs(float(head_b))
            ratio = np.abs(g["logit"][e0:e1].astype(np.float64) - og["logit"]) / np.maximum(mag, 1e-30)
            worst = max(worst, float(ratio.max()))
            assert ratio.max() <= logit_rel, (ev, float(ratio.max()))
        # chained: oracle S5 on the GPU's own logits == the GPU's track ids (bit-exact)
        tid = oracle.components(src, dst, g["logit"][e0:e1], tau, h1 - h0)
        assert np.array_equal(g["track_id"][h0:h1] - h0, tid), ev
    return worst


def _whole_batch_invariants(cfg, b, g):
    assert g["n_edges"] == g["src"].size == g["row_ptr"][-1]
    check_edge_invariants(g["src"], g["dst"], g["row_ptr"], b.plane, b.event_offsets, cfg.k, cfg.window)
    keep = g["logit"] >= oracle.logit_threshold(cfg.threshold)
    check_track_invariants(g["track_id"], g["src"], g["dst"], keep, b.event_offsets)
    assert np.isfinite(g["score"]).all() and (g["score"] >= 0).all() and (g["score"] <= 1).all()
    # CSC: a permutation of the edge ids, grouped by dst, ascending inside every group (R9, R22)
    ie, cp = g["in_edge"], g["col_ptr"]
    assert np.array_equal(np.sort(ie), np.arange(ie.size, dtype=ie.dtype))
    assert np.array_equal(np.repeat(np.arange(b.n_hits), np.diff(cp)), g["dst"][ie])
    inner = np.ones(ie.size, bool); inner[cp[:-1][np.diff(cp) > 0]] = False
    assert (np.diff(ie)[inner[1:]] > 0).all()


@pytest.mark.parametrize("name,preset", [("cfg2", "he"), ("cfg2", "parity"), ("cfg4", "parity"), ("cfg5", "parity")])
def test_full_size_bf16_invariants_and_sampled_events(name, preset):
    cfg = datagen.get_config(name)                              # bf16, 500 / 200 events: the bench configuration
    # (cfg5: the paper's operating point -- k = 50 with a radius cut, latent 32, edge encoder on [h0_src, h0_dst])
    b = datagen.generate_batch(cfg)
    if preset == "he":
        W = datagen.make_weights(cfg, "he")                     # BASELINE.json: what bench.py times
    else:
        W = centred_parity_weights(cfg, b.slice_events(0, 2))   # logits O(1): score parity is informative
    blob = datagen.pack_blob(cfg, W)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    torch.cuda.synchronize()
    _whole_batch_invariants(cfg, b, g)
    events = _sample_events(b, n_random=3 if name == "cfg2" else 1)
    if name == "cfg4":
        events = events[:3]                                     # ~9,000-hit events: the oracle takes seconds each
    if preset == "he":
        worst = _check_sampled_events(cfg, b, g, blob, "bf16", events, logit_rel=0.02)
    else:
        worst = _check_sampled_events(cfg, b, g, blob, "bf16", events, score_tol=2e-2)
        mid = np.mean((g["score"] > 0.01) & (g["score"] < 0.99))
        assert mid > 0.3, mid
    print(f"{name}/{preset}: N={b.n_hits} E={g['n_edges']} sampled events {events} "
          + (f"max |logit err| / (|w|.|e| + |b|) = {worst:.2e}" if preset == "he" else f"max|score err|={worst:.2e}"))
    if name == "cfg2":
        # track containers over the whole batch (integer work: every array equals the oracle's), and their cost
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(); t = ctx.tracks(b.n_hits, b.n_events, 3); ev1.record(); torch.cuda.synchronize()
        r = oracle.tracks(g["track_id"], b.event_offsets, 3)
        assert t["n_tracks"] == r["n_tracks"]
        for key in ("track_index", "track_offsets", "track_hits", "event_track_offsets"):
            assert np.array_equal(t[key].cpu().numpy(), r[key]), key
        print(f"{name}/{preset}: etx_tracks(min_hits=3): {r['n_tracks']} tracks, {ev0.elapsed_time(ev1):.2f} ms incl. the copies back")
    ctx.destroy()


@pytest.mark.parametrize("preset", ["parity", "he"])
def test_full_size_cfg2_every_event_chained(preset):
    # The sampled-events test above would miss a tile-scheduling fault that hits one mid-batch event, so here the
    # chained protocol runs over ALL 500 events of the headline batch at once -- the oracle is
    # OpenMP-parallel over hits / edges and needs about ten seconds: oracle S2 + S3 on the GPU's embedding == the GPU's
    # edge list; oracle S4 on those edges against every score (parity weights, 2e-2) or every logit relative to its
    # own magnitude (He weights, 0.02; R24); oracle S5 on the GPU's logits == every track id.
    cfg = datagen.get_config("cfg2")
    b = datagen.generate_batch(cfg)
    W = datagen.make_weights(cfg, "he") if preset == "he" else centred_parity_weights(cfg, b.slice_events(0, 2))
    blob = datagen.pack_blob(cfg, W)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    ctx.destroy()
    nbr, deg = oracle.knn(g["emb"], b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max)
    src, dst, _ = oracle.build_edges(nbr, deg)
    assert src.size == g["n_edges"]
    assert np.array_equal(g["src"], src) and np.array_equal(g["dst"], dst)
    o = oracle.Oracle(blob, "bf16")
    og = o.gnn(b.xyz, src, dst, want_states=(preset == "he"))
    if preset == "parity":
        err = np.abs(g["score"] - og["score"])
        worst, what = float(err.max()), "max |score err|"
        assert worst <= 2e-2, worst
        assert np.mean((g["score"] > 0.01) & (g["score"] < 0.99)) > 0.3
    else:
        _, head_w, head_b = datagen.unpack_blob(cfg, blob)[0][-1]
        assert np.isfinite(g["logit"]).all()
        mag = np.abs(og["e"]).astype(np.float32) @ np.abs(head_w[0]).astype(np.float32) + abs(float(head_b[0]))
        ratio = np.abs(g["logit"].astype(np.float64) - og["logit"]) / np.maximum(mag.astype(np.float64), 1e-30)
        worst, what = float(ratio.max()), "max |logit err| / (|w|.|e| + |b|)"
        assert worst <= 0.02, worst
    tid = oracle.components(src, dst, g["logit"], oracle.logit_threshold(cfg.threshold), b.n_hits)
    assert np.array_equal(g["track_id"], tid)
    ev_of_edge = np.searchsorted(b.event_offsets, src, side="right") - 1
    print(f"cfg2/{preset}: {b.n_events}/{b.n_events} events compared element by element (N={b.n_hits}, E={src.size}, "
          f"{np.unique(ev_of_edge).size} events with edges): edges and track ids equal, {what} = {worst:.3e}")


def test_full_size_fp32_cfg1_end_to_end_sampled_events():
    cfg = datagen.get_config("cfg1")                            # 64 events, fp32 throughout
    b = datagen.generate_batch(cfg)
    W = centred_parity_weights(cfg, b.slice_events(0, 2))
    blob = datagen.pack_blob(cfg, W)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    _whole_batch_invariants(cfg, b, g)
    worst = _check_sampled_events(cfg, b, g, blob, "fp32", _sample_events(b, 2), score_tol=1e-4)
    print(f"cfg1/fp32: N={b.n_hits} E={g['n_edges']} max|score err|={worst:.2e}")
    ctx.destroy()


@pytest.mark.parametrize("name", ["cfg3", "cfg3b"])          # state stored as fp32 (cfg 3) and as bf16 (cfg 3b)
def test_full_size_int8_cfg3_bit_exact_on_sampled_events(name):
    # 1000 events, INT8 MLPs (R21): integer accumulation is order-free and every other op is a single pinned fp32
    # op, so on sampled events the embedding, the edges, the logits and the track ids must equal the oracle's bits
    cfg = datagen.get_config(name)
    b = datagen.generate_batch(cfg)
    W = centred_parity_weights(cfg.replace(precision="fp32"), b.slice_events(0, 2))
    cal = datagen.generate_batch(datagen.get_config("cfg1"), n_events=datagen.configs.CALIBRATION_EVENTS,
                                 seed=datagen.configs.CALIBRATION_SEED)
    scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), cal.xyz, cal.plane, cal.event_offsets, cfg.k, cfg.window)
    blob = datagen.pack_blob(cfg, W, scales)
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    _whole_batch_invariants(cfg, b, g)
    o = oracle.Oracle(blob, "int8", state_dtype=cfg.state_dtype)      # cfg 3b stores the state as bf16 (R21)
    eo, rp = b.event_offsets, g["row_ptr"]
    events = _sample_events(b, n_random=2)
    for ev in events:
        h0, h1 = int(eo[ev]), int(eo[ev + 1])
        e0, e1 = int(rp[h0]), int(rp[h1])
        sub = b.slice_events(ev, ev + 1)
        r = o.run(sub.xyz, sub.plane, sub.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
        assert np.array_equal(g["emb"][h0:h1], r["emb"]), ev
        assert np.array_equal(g["src"][e0:e1] - h0, r["src"]) and np.array_equal(g["dst"][e0:e1] - h0, r["dst"]), ev
        assert np.array_equal(g["logit"][e0:e1], r["logit"]), ev
        assert np.abs(g["score"][e0:e1] - r["score"]).max(initial=0.0) <= 1e-4
        assert np.array_equal(g["track_id"][h0:h1] - h0, r["track_id"]), ev
    print(f"{name}/int8 (state {cfg.state_dtype}): N={b.n_hits} E={g['n_edges']} sampled events {events} bit-exact")
    ctx.destroy()
