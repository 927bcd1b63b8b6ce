"""Hyper-parameter presets: BASELINE.json `configs[0..4]`, restated.

PAPER.md gives the structure (26 planes L26; k_max-NN over the next planes
L101; n message-passing steps with distinct weights L148; threshold L80); the
concrete sizes below are BASELINE.json's, because the paper does not state the
embedding MLP's shape and the configs choose their own
k, w, d, L.
"""
from __future__ import annotations

import dataclasses
import math
from dataclasses import dataclass

N_PLANES = 26
PLANE_Z0, PLANE_DZ = -300.0, 42.0  # BASELINE.json cfg 0: z_i = -300 + 42 i
NORM_OFFSET = (0.0, 0.0, 300.0)    # features (x/40, y/40, (z+300)/1050)
NORM_DIV = (40.0, 40.0, 1050.0)
CYL_OFFSET = (-20.0, 0.0, 300.0)   # cylindrical embedding input ((r-20)/12, phi/pi, (z+300)/1050): DESIGN.md R27
CYL_DIV = (12.0, 3.14159274, 1050.0)


@dataclass(frozen=True)
class EtxConfig:
    name: str
    # --- event generator -------------------------------------------------
    n_events: int
    fixed_pv: int | None        # exact number of PVs (cfg 0) or None -> Poisson(mu_pv)
    mu_pv: float
    fixed_tracks: int | None    # exact tracks per PV (cfg 0) or None -> Poisson(mu_tracks)
    mu_tracks: float
    noise_frac: float           # Poisson(noise_frac * n_signal(event, plane)) noise hits
    events_seed: int
    # --- model -----------------------------------------------------------
    emb_hidden: int
    emb_n_hidden_layers: int
    emb_dim: int
    k: int
    window: int
    d2_max: float
    gnn_latent: int
    gnn_iters: int
    threshold: float
    precision: str              # "fp32" | "bf16" | "int8"
    edge_enc_input: int = 0     # 0: |f_dst - f_src| (configs), 1: [h0_src, h0_dst]
    emb_input: int = 0          # 0: the embedding reads the Cartesian features, 1: normalised (r, phi, z) (L96, R27)
    weights_seed: int = 7
    state_dtype: str = "auto"   # storage of h, e, m: "auto" (fp32 for fp32 / int8, bf16 for bf16), "fp32", "bf16" (int8 only; R21)
    triplets: int = 0           # 1: the blob also carries the two triplet classifiers (R28)
    triplet_threshold: float = 0.5

    def replace(self, **kw) -> "EtxConfig":
        return dataclasses.replace(self, **kw)


_COMMON = dict(emb_dim=4, d2_max=math.inf, threshold=0.5)

CONFIGS: dict[str, EtxConfig] = {
    # cfg 0: one small event, fp32
    "cfg0": EtxConfig(name="cfg0", n_events=1, fixed_pv=1, mu_pv=1.0, fixed_tracks=20,
                      mu_tracks=20.0, noise_frac=0.0, events_seed=1000,
                      emb_hidden=64, emb_n_hidden_layers=2, k=4, window=1,
                      gnn_latent=32, gnn_iters=4, precision="fp32", **_COMMON),
    # cfg 1: 64 events at nominal pile-up, fp32
    "cfg1": EtxConfig(name="cfg1", n_events=64, fixed_pv=None, mu_pv=5.0, fixed_tracks=None,
                      mu_tracks=40.0, noise_frac=0.02, events_seed=1001,
                      emb_hidden=128, emb_n_hidden_layers=3, k=10, window=2,
                      gnn_latent=64, gnn_iters=6, precision="fp32", **_COMMON),
    # cfg 2 (headline): 500 events, bf16 MLPs
    "cfg2": EtxConfig(name="cfg2", n_events=500, fixed_pv=None, mu_pv=5.0, fixed_tracks=None,
                      mu_tracks=40.0, noise_frac=0.02, events_seed=1002,
                      emb_hidden=128, emb_n_hidden_layers=3, k=10, window=2,
                      gnn_latent=64, gnn_iters=6, precision="bf16", **_COMMON),
    # cfg 3: 1000 events, INT8 MLPs, h / e / m stored as fp32 (the INT8 configuration as round 1 measured it, so that
    # its row stays comparable from round to round)
    "cfg3": EtxConfig(name="cfg3", n_events=1000, fixed_pv=None, mu_pv=5.0, fixed_tracks=None,
                      mu_tracks=40.0, noise_frac=0.02, events_seed=1003,
                      emb_hidden=128, emb_n_hidden_layers=3, k=10, window=2,
                      gnn_latent=64, gnn_iters=6, precision="int8", **_COMMON),
    # cfg 3b: the same events and arithmetic with h, e, m stored as bf16 (R21: the config text fixes the
    # arithmetic -- int8 operands, int32 accumulation, fp32 dequantisation -- not the storage of the state).  Its scores
    # differ from cfg 3's (the state is rounded on store), which is why it has a name of its own.
    "cfg3b": EtxConfig(name="cfg3b", n_events=1000, fixed_pv=None, mu_pv=5.0, fixed_tracks=None,
                       mu_tracks=40.0, noise_frac=0.02, events_seed=1003,
                       emb_hidden=128, emb_n_hidden_layers=3, k=10, window=2,
                       gnn_latent=64, gnn_iters=6, precision="int8", state_dtype="bf16", **_COMMON),
    # cfg 4: high-occupancy stress, bf16
    "cfg4": EtxConfig(name="cfg4", n_events=200, fixed_pv=None, mu_pv=20.0, fixed_tracks=None,
                      mu_tracks=40.0, noise_frac=0.02, events_seed=1004,
                      emb_hidden=128, emb_n_hidden_layers=3, k=16, window=3,
                      gnn_latent=64, gnn_iters=8, precision="bf16", **_COMMON),
    # cfg 5 (not in BASELINE.json; SURVEY.md sec. 8(f) "next", item 1): the paper's own operating point -- k_max = 50
    # with a radius cut, w = 2, latent 32, n = 5 steps with distinct weights (L148), edge encoder on
    # [h0_src, h0_dst] (L133).  The paper's d2_max = 0.9 only means something for its trained embedding; with
    # seeded random weights the cut is set to the value that leaves ~14 edges per hit (L74: ~30,000 edges for
    # ~2,200 hits), measured on six events of this generator with the oracle.  On those six events 0.06 % of the
    # hits fill all 50 slots (the paper reports < 0.1 %, L257); over the first 24 events it is 3 %, because the busiest
    # events (> 4,500 hits) saturate 10-20 % of their hits -- a fixed cut on an untrained embedding tracks density.  Embedding shape as cfg 2, input the paper's normalised cylindrical
    # coordinates (L96, R27).
    "cfg5": EtxConfig(name="cfg5", n_events=500, fixed_pv=None, mu_pv=5.0, fixed_tracks=None,
                      mu_tracks=40.0, noise_frac=0.02, events_seed=1005,
                      emb_hidden=128, emb_n_hidden_layers=3, emb_dim=4, k=50, window=2, d2_max=0.154,
                      gnn_latent=32, gnn_iters=5, threshold=0.5, precision="bf16", edge_enc_input=1, emb_input=1),
}

CALIBRATION_SEED = 99      # 16-event calibration batch for INT8 (cfg-1 generator)
CALIBRATION_EVENTS = 16


def get_config(name: str) -> EtxConfig:
    return CONFIGS[name]
