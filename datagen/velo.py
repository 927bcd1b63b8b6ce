"""Seeded synthetic VELO-shaped events (stand-in for the LHCb simulation of
PAPER.md L62, which is not available).  The recipe is BASELINE.json's config
text with the readings of SURVEY.md section 8(c) A23, restated in DESIGN.md section 5:

* 26 planes at z_i = -300 + 42 i mm, acceptance annulus 5.1 <= r <= 42 mm.
* primary vertices at (N(0,.05), N(0,.05), N(0,50)) mm; straight forward
  tracks, eta ~ U[2,5], phi ~ U[0,2pi), slope tan(2 atan(exp(-eta))).
* one hit per plane with z > z_PV whose (unsmeared) crossing point is inside
  the annulus, kept with probability 0.98, x and y smeared by N(0, 0.012) mm.
* noise: Poisson(noise_frac * n_signal(event, plane)) hits per (event, plane),
  uniform in area on the annulus.
* hits ordered by event, then plane, then atan2(y, x) (stable).

Only numpy's counter-based Philox generator is used, keyed by (seed, event),
so every event can be regenerated independently.  No method arithmetic here.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .configs import N_PLANES, PLANE_DZ, PLANE_Z0, EtxConfig

R_MIN, R_MAX = 5.1, 42.0
HIT_EFF = 0.98
SMEAR_MM = 0.012


@dataclass
class EventBatch:
    xyz: np.ndarray            # [N,3] float32, mm
    plane: np.ndarray          # [N]   int32, 0..25
    event_offsets: np.ndarray  # [B+1] int32
    particle: np.ndarray       # [N]   int64: event-local particle id, -1 for noise (truth, host only)

    @property
    def n_hits(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def n_events(self) -> int:
        return int(self.event_offsets.shape[0] - 1)

    def slice_events(self, b0: int, b1: int) -> "EventBatch":
        """Events [b0, b1) as a batch of their own (offsets rebased)."""
        o = self.event_offsets
        lo, hi = int(o[b0]), int(o[b1])
        return EventBatch(self.xyz[lo:hi].copy(), self.plane[lo:hi].copy(),
                          (o[b0:b1 + 1] - o[b0]).astype(np.int32), self.particle[lo:hi].copy())


def _one_event(seed: int, index: int, cfg: EtxConfig):
    rng = np.random.Generator(np.random.Philox(key=[seed & 0xFFFFFFFFFFFFFFFF, index]))
    n_pv = cfg.fixed_pv if cfg.fixed_pv is not None else int(rng.poisson(cfg.mu_pv))
    pv = np.stack([rng.normal(0.0, 0.05, n_pv), rng.normal(0.0, 0.05, n_pv),
                   rng.normal(0.0, 50.0, n_pv)], axis=1) if n_pv else np.zeros((0, 3))
    if cfg.fixed_tracks is not None:
        n_trk = np.full(n_pv, cfg.fixed_tracks, dtype=np.int64)
    else:
        n_trk = rng.poisson(cfg.mu_tracks, n_pv).astype(np.int64)
    T = int(n_trk.sum())
    origin = np.repeat(pv, n_trk, axis=0)                       # [T,3]
    eta = rng.uniform(2.0, 5.0, T)
    phi = rng.uniform(0.0, 2.0 * np.pi, T)
    slope = np.tan(2.0 * np.arctan(np.exp(-eta)))               # dr/dz, forward tracks only
    zp = PLANE_Z0 + PLANE_DZ * np.arange(N_PLANES)              # [P]
    dz = zp[None, :] - origin[:, 2:3]                           # [T,P]
    x = origin[:, 0:1] + dz * (slope * np.cos(phi))[:, None]
    y = origin[:, 1:2] + dz * (slope * np.sin(phi))[:, None]
    r = np.hypot(x, y)
    in_acc = (dz > 0.0) & (r >= R_MIN) & (r <= R_MAX)           # tested before smearing
    keep = in_acc & (rng.random((T, N_PLANES)) < HIT_EFF)
    x = x + rng.normal(0.0, SMEAR_MM, (T, N_PLANES))
    y = y + rng.normal(0.0, SMEAR_MM, (T, N_PLANES))
    t_idx, p_idx = np.nonzero(keep)
    sx, sy, sp, spid = x[t_idx, p_idx], y[t_idx, p_idx], p_idx.astype(np.int64), t_idx.astype(np.int64)
    # noise hits
    n_sig = np.bincount(sp, minlength=N_PLANES)
    n_noise = rng.poisson(cfg.noise_frac * n_sig) if cfg.noise_frac > 0 else np.zeros(N_PLANES, np.int64)
    tot = int(n_noise.sum())
    if tot:
        rr = np.sqrt(rng.uniform(R_MIN ** 2, R_MAX ** 2, tot))
        ph = rng.uniform(0.0, 2.0 * np.pi, tot)
        nx, ny = rr * np.cos(ph), rr * np.sin(ph)
        npl = np.repeat(np.arange(N_PLANES), n_noise)
        sx = np.concatenate([sx, nx]); sy = np.concatenate([sy, ny])
        sp = np.concatenate([sp, npl]); spid = np.concatenate([spid, np.full(tot, -1, np.int64)])
    # order: plane, then azimuth, ties by generation order (stable sorts)
    az = np.arctan2(sy, sx)
    order = np.argsort(az, kind="stable")
    order = order[np.argsort(sp[order], kind="stable")]
    sx, sy, sp, spid = sx[order], sy[order], sp[order], spid[order]
    xyz = np.stack([sx, sy, zp[sp]], axis=1).astype(np.float32) if sx.size else np.zeros((0, 3), np.float32)
    return xyz, sp.astype(np.int32), spid


def generate_batch(cfg: EtxConfig, n_events: int | None = None, seed: int | None = None,
                   first_event: int = 0) -> EventBatch:
    """Events first_event .. first_event+n_events-1 of the stream (seed, cfg)."""
    n_events = cfg.n_events if n_events is None else n_events
    seed = cfg.events_seed if seed is None else seed
    xs, ps, ids, off = [], [], [], [0]
    for b in range(n_events):
        xyz, pl, pid = _one_event(seed, first_event + b, cfg)
        xs.append(xyz); ps.append(pl); ids.append(pid)
        off.append(off[-1] + xyz.shape[0])
    return EventBatch(np.concatenate(xs, axis=0) if xs else np.zeros((0, 3), np.float32),
                      np.concatenate(ps) if ps else np.zeros(0, np.int32),
                      np.asarray(off, dtype=np.int32),
                      np.concatenate(ids) if ids else np.zeros(0, np.int64))


def hand_batch(events: list[list[tuple[float, float, int]]]) -> EventBatch:
    """A batch from hand-written events: each event a list of (x_mm, y_mm, plane),
    which must already be sorted by plane.  z is the plane's z.  For fixtures."""
    xs, ps, off = [], [], [0]
    for ev in events:
        for (x, y, p) in ev:
            xs.append((x, y, PLANE_Z0 + PLANE_DZ * p)); ps.append(p)
        off.append(len(ps))
    xyz = np.asarray(xs, dtype=np.float32).reshape(-1, 3)
    return EventBatch(xyz, np.asarray(ps, dtype=np.int32), np.asarray(off, dtype=np.int32),
                      np.full(len(ps), -1, np.int64))
