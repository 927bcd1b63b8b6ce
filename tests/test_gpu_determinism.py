"""Determinism soak (stands in for compute-sanitizer racecheck, which is closed on this pool): the lock-free union-find,
the CSC bucket walk, the k-NN insertion and the warp-specialised tensor-core pipelines are run many times on the same
input; every output array must come out bit-identical every time (no atomics on floating point, min-index
roots, ascending-edge-id sums).  The first run's arrays are also checked against the oracle-independent invariants."""
import hashlib

import numpy as np
import pytest
import torch

import datagen
from gpu_utils import dev, make_ctx
from helpers import check_edge_invariants

pytestmark = pytest.mark.gpu


def _digest(ctx, out, n_hits, extra=("row_ptr", "col_ptr", "in_edge")):
    r = ctx.results(out)
    h = hashlib.sha256()
    for key in ("src", "dst", "logit", "score", "track_id"):
        h.update(r[key].cpu().numpy().tobytes())
    for name in extra:
        h.update(ctx.buffer(name, torch.int32).cpu().numpy().tobytes())
    return h.hexdigest(), r


@pytest.mark.parametrize("name,precision,n_events,reps", [("cfg2", "bf16", 500, 12), ("cfg1", "fp32", 8, 60), ("cfg3", "int8", 40, 25), ("cfg3b", "int8", 40, 25),
                                                          ("cfg5", "bf16", 60, 25), ("cfg4", "bf16", 6, 25)])
def test_repeated_runs_are_bit_identical(name, precision, n_events, reps):
    cfg = datagen.get_config(name).replace(precision=precision)
    b = datagen.generate_batch(cfg, n_events=n_events)
    W = datagen.make_weights(cfg, "parity")
    scales = None
    if precision == "int8":
        import oracle
        cal = datagen.generate_batch(datagen.get_config("cfg1"), n_events=4, seed=datagen.configs.CALIBRATION_SEED)
        scales = oracle.calibrate_int8(datagen.pack_blob(cfg, W), cal.xyz, cal.plane, cal.event_offsets, cfg.k, cfg.window, cfg.d2_max)
    ctx = make_ctx(cfg, datagen.pack_blob(cfg, W, scales), b)
    xyz, plane = dev(b.xyz), dev(b.plane)
    first, r0 = _digest(ctx, ctx.run(xyz, plane, b.event_offsets), b.n_hits)
    rp = ctx.buffer("row_ptr", torch.int32).cpu().numpy()
    check_edge_invariants(r0["src"].cpu().numpy(), r0["dst"].cpu().numpy(), rp, b.plane, b.event_offsets, cfg.k, cfg.window)
    for i in range(reps):
        d, _ = _digest(ctx, ctx.run(xyz, plane, b.event_offsets), b.n_hits)
        assert d == first, f"run {i + 1} differs from run 0"
    # a second handle on a second stream, running concurrently with the first, gives the same bits
    ctx2 = make_ctx(cfg, datagen.pack_blob(cfg, W, scales), b)
    s2 = torch.cuda.Stream()
    with torch.cuda.stream(s2):
        out2 = ctx2.run(xyz, plane, b.event_offsets)
    out1 = ctx.run(xyz, plane, b.event_offsets)
    torch.cuda.synchronize()
    assert _digest(ctx2, out2, b.n_hits)[0] == first and _digest(ctx, out1, b.n_hits)[0] == first
    ctx.destroy(); ctx2.destroy()
