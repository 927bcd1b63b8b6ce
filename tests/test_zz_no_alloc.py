"""etx_tracks_static -- the track regrouping for callers that may not allocate device memory -- against etx_tracks.

Some users of this library run inside a host framework that owns every byte of device memory and forbids cudaMalloc /
cudaFree once its event loop has started (the paper's target, Allen, is one: PAPER.md L223), or are plug-ins that
receive raw device pointers and no allocator.  They cannot create a handle (etx_create allocates the workspace), so
etx_tracks is closed to them.  etx_tracks_static takes its work arrays from a fixed array inside libetx.so instead
(include/etx.h: at most ETX_TRACKS_STATIC_MAX_HITS hits, all calls on a GPU share the array).

What is checked: on the GPU's own track ids, every output array of the new call equals the existing path's (integer
work: the tolerance of the other track-container tests, i.e. none), on two calls in a row with different batches -- the
second smaller than the first, so that it runs over whatever the first left in the shared array -- then the first again;
sizes beyond the maximum are refused with a message; the calls leave the device's free memory where it was.

The file is named so that pytest collects it last: `-x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process and after the other tests (nothing else touches the array).
"""
import numpy as np
import pytest
import torch

import datagen
import paper_2407_12119_b200 as etx
from gpu_utils import dev, make_ctx, run_gpu
from helpers import centred_parity_weights

pytestmark = pytest.mark.gpu
KEYS = ("track_index", "track_offsets", "track_hits", "event_track_offsets")


def _existing_path(name, n_events, precision, min_hits, seed=None):
    """Run the pipeline and etx_tracks (the handle's own workspace); returns the batch, the track ids and its result."""
    cfg = datagen.get_config(name).replace(precision=precision)
    b = datagen.generate_batch(cfg, n_events=n_events, seed=seed)
    # weights whose scores straddle the threshold (bias centred on the first events), so that tracks of many sizes exist
    blob = datagen.pack_blob(cfg, centred_parity_weights(cfg, b.slice_events(0, min(2, b.n_events))))
    ctx = make_ctx(cfg, blob, b)
    g = run_gpu(ctx, b, debug=False)
    t = ctx.tracks(b.n_hits, b.n_events, min_hits)
    want = {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in t.items()}
    ctx.destroy()
    return b, g["track_id"], want


def _caller_buffers(n_hits, n_events):
    """The caller's output buffers, filled with a pattern so that an element the call fails to write shows up."""
    i32 = dict(dtype=torch.int32, device="cuda")
    return dict(track_index=torch.full((n_hits,), -7, **i32), track_offsets=torch.full((n_hits + 1,), -7, **i32),
                track_hits=torch.full((n_hits,), -7, **i32), event_track_offsets=torch.full((n_events + 1,), -7, **i32),
                n_tracks=torch.full((1,), -7, **i32))


def _check(out, want, what):
    torch.cuda.synchronize()
    T = int(out["n_tracks"].item())
    assert T == want["n_tracks"] and T > 0, what
    offs = out["track_offsets"].cpu().numpy()
    assert np.array_equal(offs[:T + 1], want["track_offsets"]), what
    assert np.all(offs[T:] == offs[T]), what                                  # entries past n_tracks repeat the total
    assert np.array_equal(out["track_index"].cpu().numpy(), want["track_index"]), what
    assert np.array_equal(out["track_hits"].cpu().numpy()[:offs[T]], want["track_hits"]), what
    assert np.array_equal(out["event_track_offsets"].cpu().numpy(), want["event_track_offsets"]), what


def test_tracks_static_equals_etx_tracks_on_consecutive_calls_and_allocates_nothing():
    big = _existing_path("cfg1", 5, "fp32", 3)
    small = _existing_path("cfg0", 1, "fp32", 4, seed=11)
    assert small[0].n_hits < big[0].n_hits
    cases = []
    for (b, tid, want), min_hits in ((big, 3), (small, 4)):
        cases.append((dev(tid, torch.int32), dev(np.asarray(b.event_offsets, np.int32)), min_hits,
                      _caller_buffers(b.n_hits, b.n_events), want))
    torch.cuda.synchronize()
    # two calls in a row (big, then small over the big one's leftovers), with no synchronisation in between: the stream
    # orders them, as the header asks
    for tid, eo, min_hits, out, _ in cases:
        etx.tracks_static(tid, eo, min_hits, out)
    for i, (_, _, _, out, want) in enumerate(cases):
        _check(out, want, f"call {i}")
    # and again, now that every kernel of the call has been loaded: device memory in use must not move
    free_before, _ = torch.cuda.mem_get_info()
    for tid, eo, min_hits, out, want in cases:
        for key in out:
            out[key].fill_(-7)
        etx.tracks_static(tid, eo, min_hits, out)
        _check(out, want, "repeat")
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before


def test_tracks_static_at_the_headline_batch_size():
    # cfg 2 as bench.py runs it: 500 events, 1,042,793 hits -- 99.4 % of ETX_TRACKS_STATIC_MAX_HITS, 510 blocks of the
    # prefix sums -- twice in a row with different filters
    b, tid, want3 = _existing_path("cfg2", None, "bf16", 3)
    assert 0.9 * etx.TRACKS_STATIC_MAX_HITS < b.n_hits <= etx.TRACKS_STATIC_MAX_HITS
    d_tid, d_eo = dev(tid, torch.int32), dev(np.asarray(b.event_offsets, np.int32))
    out3, out1 = _caller_buffers(b.n_hits, b.n_events), _caller_buffers(b.n_hits, b.n_events)
    etx.tracks_static(d_tid, d_eo, 3, out3)
    etx.tracks_static(d_tid, d_eo, 1, out1)
    _check(out3, want3, "min_hits 3")
    # min_hits = 1: every hit is in a track, tracks are the components in ascending order of their smallest hit
    T = int(out1["n_tracks"].item())
    roots = np.flatnonzero(tid == np.arange(tid.size))
    assert T == roots.size
    idx = out1["track_index"].cpu().numpy()
    assert np.array_equal(idx, np.searchsorted(roots, tid))
    offs = out1["track_offsets"].cpu().numpy()
    assert offs[T] == b.n_hits and np.array_equal(np.diff(offs[:T + 1]), np.bincount(idx, minlength=T))
    hits = out1["track_hits"].cpu().numpy()
    assert np.array_equal(hits, np.argsort(idx, kind="stable"))               # grouped by track, ascending inside


def test_tracks_static_refuses_what_does_not_fit_and_handles_empty_input():
    n = etx.TRACKS_STATIC_MAX_HITS + 1
    tid = torch.zeros(n, dtype=torch.int32, device="cuda")
    eo = torch.tensor([0, n], dtype=torch.int32, device="cuda")
    out = _caller_buffers(n, 1)
    with pytest.raises(etx.EtxError) as ei:
        etx.tracks_static(tid, eo, 3, out)
    assert ei.value.status == -3 and "ETX_TRACKS_STATIC_MAX_HITS" in str(ei.value)
    torch.cuda.synchronize()
    assert int(out["n_tracks"].item()) == -7                                   # nothing was launched
    with pytest.raises(etx.EtxError) as ei:
        etx.tracks_static(tid[:8], eo, 0, _caller_buffers(8, 1))               # min_hits < 1
    assert ei.value.status == -1
    # no hits at all: zero tracks, all-zero event offsets
    out = _caller_buffers(0, 2)
    etx.tracks_static(tid[:0], torch.zeros(3, dtype=torch.int32, device="cuda"), 3, out)
    torch.cuda.synchronize()
    assert int(out["n_tracks"].item()) == 0 and int(out["track_offsets"][0].item()) == 0
    assert np.array_equal(out["event_track_offsets"].cpu().numpy(), np.zeros(3, np.int32))
