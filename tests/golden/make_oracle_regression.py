"""Writes tests/golden/oracle_regression.json: digests of what the oracle computes on three small seeded inputs.

This is a regression pin, not an independent one (those are in tests/test_oracle_pins.py): it calls only `oracle/`
and `datagen/`, never the CUDA path, and freezes the oracle's bits so that a later change to its arithmetic, its
compiler flags or the input generator cannot go unnoticed.  Such a change has to regenerate this file in the same
commit and name, in the commit message, the passage of PAPER.md or the DESIGN.md reading that justifies it.

    python tests/golden/make_oracle_regression.py
"""
import hashlib
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import datagen  # noqa: E402
import oracle  # noqa: E402

CASES = [("cfg0", 1, "fp32", "parity", {}), ("cfg1", 2, "fp32", "he", {}), ("cfg1", 2, "bf16", "he", {}),
         ("cfg5", 1, "bf16", "parity", {}), ("cfg1", 2, "fp32", "he", {"edge_enc_input": 1, "emb_input": 1})]


def digest(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()[:24]


def compute():
    out = []
    for name, n_events, precision, preset, extra in CASES:
        cfg = datagen.get_config(name).replace(precision=precision, **extra)
        b = datagen.generate_batch(cfg, n_events=n_events)
        blob = datagen.pack_blob(cfg, datagen.make_weights(cfg, preset))
        r = oracle.Oracle(blob, precision).run(b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
        t = oracle.tracks(r["track_id"], b.event_offsets, 3)
        out.append(dict(case=[name, n_events, precision, preset, extra], n_hits=int(b.n_hits), n_edges=int(r["src"].size),
                        n_tracks=int(t["n_tracks"]), xyz=digest(b.xyz), emb=digest(r["emb"]), src=digest(r["src"]),
                        dst=digest(r["dst"]), logit=digest(r["logit"]), track_id=digest(r["track_id"]),
                        logit_head=[float(x).hex() for x in r["logit"][:4]]))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")
    with open(path, "w") as f:
        json.dump(compute(), f, indent=1)
    print("wrote", path)
