"""Helpers for the -m gpu parity tests: run the C-ABI library through its Python binding and bring
results back as numpy arrays.  The expected values always come from oracle/ (never from the GPU)."""
from __future__ import annotations

import numpy as np
import torch

import datagen
import paper_2407_12119_b200 as etx


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def make_ctx(cfg, blob, batch=None, precision=None, engine="auto", max_events=None, max_hits=None, validate=False,
             max_triplets=0):
    B = max_events if max_events is not None else max(batch.n_events, 1)
    N = max_hits if max_hits is not None else max(batch.n_hits, 1)
    hp = etx.hyperparams_from_config(cfg, B, N, precision=precision, engine=engine, validate_input=validate,
                                     max_triplets=max_triplets)
    return etx.Etx(blob, hp)


def run_gpu(ctx, batch, emb=None, src=None, dst=None, logit=None, last_stage=5, debug=True):
    xyz, plane = dev(batch.xyz), dev(batch.plane)
    kw = {}
    if emb is not None:
        kw["emb"] = dev(np.asarray(emb, np.float32))
    if src is not None:
        kw["src"], kw["dst"] = dev(np.asarray(src, np.int32)), dev(np.asarray(dst, np.int32))
    if logit is not None:
        kw["logit"] = dev(np.asarray(logit, np.float32))
    if debug or kw or last_stage != 5:
        out = ctx.dbg_run(xyz, plane, batch.event_offsets, last_stage=last_stage, **kw)
    else:
        out = ctx.run(xyz, plane, batch.event_offsets)
    r = ctx.results(out)
    res = {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in r.items()}
    N = batch.n_hits
    res["emb"] = ctx.buffer("emb", torch.float32).cpu().numpy().reshape(N, 4)
    if last_stage >= 2:
        res["row_ptr"] = ctx.buffer("row_ptr", torch.int32).cpu().numpy()
    if last_stage >= 3:
        res["col_ptr"] = ctx.buffer("col_ptr", torch.int32).cpu().numpy()
        res["in_edge"] = ctx.buffer("in_edge", torch.int32).cpu().numpy()
    return res


def state(ctx, name, rows, d):
    """h / e / m as float32 numpy [rows, d] whatever the state dtype."""
    bf16 = ctx.hp.precision == 1 or (ctx.hp.precision == 2 and ctx.hp.state_dtype == 2)
    t = ctx.buffer(name, torch.bfloat16 if bf16 else torch.float32)
    return t.float().cpu().numpy().reshape(rows, d)
