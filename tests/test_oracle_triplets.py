"""Pins for the oracle's triplet stage (sec. 5.3, sec. 5.4; R28-R31): brute-force
enumeration over all pairs of edges, an independent set / BFS formulation of the four track-building phases,
hand-built fixtures (an e+e- like pair sharing its first hits, skipped planes), float64 / torch-bfloat16
restatements of the classifier, invariants.  CPU only."""
import itertools

import numpy as np
import pytest
import torch

import datagen
import oracle
from helpers import centred_parity_weights, f32_chain, torch_bf16, toy_config

F = np.float32


def _random_graph(seed, n=14, E=40, n_planes=5):
    rng = np.random.default_rng(seed)
    plane = np.sort(rng.integers(0, n_planes, n)).astype(np.int32)
    pairs = set()
    while len(pairs) < E:
        a, b = rng.integers(0, n, 2)
        if plane[a] < plane[b]:
            pairs.add((int(a), int(b)))
    pairs = sorted(pairs)                                     # src-sorted, distinct (as S3 builds them)
    src = np.array([p[0] for p in pairs], np.int32); dst = np.array([p[1] for p in pairs], np.int32)
    keep = (rng.random(len(pairs)) < 0.7).astype(np.uint8)
    return plane, src, dst, keep


def _triplets_bruteforce(src, dst, keep, kind):
    """All ordered pairs of kept edges, classified by which end they share (L154-158)."""
    out = []
    E = src.size
    for i, j in itertools.product(range(E), range(E)):
        if i == j or not keep[i] or not keep[j]:
            continue
        if kind == "articulation" and dst[i] == src[j]:
            out.append((int(dst[i]), i, j))
        if kind == "left_elbow" and src[i] == src[j] and i < j:
            out.append((int(src[i]), i, j))
        if kind == "right_elbow" and dst[i] == dst[j] and i < j:
            out.append((int(dst[i]), i, j))
    out.sort()                                                # R29: common hit, first, second
    return out


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_triplets_equal_bruteforce_over_all_edge_pairs(seed):
    plane, src, dst, keep = _random_graph(seed)
    n = plane.size
    total = 0
    for kind in ("articulation", "left_elbow", "right_elbow"):
        f, s, h = oracle.triplets(src, dst, keep, n, kind)
        want = _triplets_bruteforce(src, dst, keep, kind)
        assert [(int(c), int(a), int(b)) for a, b, c in zip(f, s, h)] == want, kind
        total += len(want)
        # invariants: kept edges only, exactly one common hit of the stated kind, three distinct hits
        assert keep[f].all() and keep[s].all()
        if kind == "articulation":
            assert np.array_equal(dst[f], h) and np.array_equal(src[s], h)
            assert (plane[src[f]] < plane[h]).all() and (plane[h] < plane[dst[s]]).all()
        elif kind == "left_elbow":
            assert np.array_equal(src[f], h) and np.array_equal(src[s], h) and (f < s).all() and (dst[f] != dst[s]).all()
        else:
            assert np.array_equal(dst[f], h) and np.array_equal(dst[s], h) and (f < s).all() and (src[f] != src[s]).all()
    assert total > 20
    # closed form of the counts: sum over hits of in*out, C(out,2), C(in,2) of the kept degrees
    od = np.bincount(src[keep > 0], minlength=n); idg = np.bincount(dst[keep > 0], minlength=n)
    assert oracle.triplets(src, dst, keep, n, "articulation")[0].size == int((od * idg).sum())
    assert oracle.triplets(src, dst, keep, n, "left_elbow")[0].size == int((od * (od - 1) // 2).sum())
    assert oracle.triplets(src, dst, keep, n, "right_elbow")[0].size == int((idg * (idg - 1) // 2).sum())


def test_triplets_edge_cases():
    e = np.zeros(0, np.int32)
    for kind in ("articulation", "left_elbow", "right_elbow"):
        f, s, h = oracle.triplets(e, e, np.zeros(0, np.uint8), 5, kind)
        assert f.size == s.size == h.size == 0
    src = np.array([0, 0, 1], np.int32); dst = np.array([1, 2, 2], np.int32)
    none = np.zeros(3, np.uint8)
    assert oracle.triplets(src, dst, none, 3, "articulation")[0].size == 0     # nothing kept: no triplets (L146)
    allk = np.ones(3, np.uint8)
    assert [x.tolist() for x in oracle.triplets(src, dst, allk, 3, "articulation")] == [[0], [2], [1]]
    assert [x.tolist() for x in oracle.triplets(src, dst, allk, 3, "left_elbow")] == [[0], [1], [0]]
    assert [x.tolist() for x in oracle.triplets(src, dst, allk, 3, "right_elbow")] == [[1], [2], [2]]


# ------------------------------------------------------------------ the classifier (L80, L160; R28)
def _triplet_model(precision="fp32", d=16):
    cfg = toy_config(d=d, L=1, precision=precision).replace(triplets=1)
    W = datagen.make_weights(cfg, "parity", seed=3)
    return cfg, W, datagen.pack_blob(cfg, W)


def test_triplet_classifier_equals_float64_and_pinned_fp32_restatement():
    cfg, W, blob = _triplet_model()
    lay = {n: (w, b) for n, w, b in W}
    rng = np.random.default_rng(4)
    e = rng.normal(0, 1, (30, 16)).astype(F)
    first = rng.integers(0, 30, 50).astype(np.int32); second = rng.integers(0, 30, 50).astype(np.int32)
    o = oracle.Oracle(blob, "fp32")
    assert o.has_triplets()
    for elbow, (n0, n1) in ((False, ("tart0", "tart1")), (True, ("telb0", "telb1"))):
        z, sc = o.triplet_scores(e, first, second, elbow)
        x = np.concatenate([e[first], e[second]], 1)                         # [e_first, e_second]: order matters
        ref = f32_chain(np.maximum(f32_chain(x, *lay[n0]), 0), *lay[n1])[:, 0]
        assert np.array_equal(z.view(np.uint32), ref.view(np.uint32))
        x64 = x.astype(np.float64)
        z64 = np.maximum(x64 @ lay[n0][0].T.astype(np.float64) + lay[n0][1], 0) @ lay[n1][0][0].astype(np.float64) + lay[n1][1][0]
        assert np.abs(z - z64).max() < 1e-4 and np.abs(z64).max() > 0.1
        assert np.abs(sc - 1 / (1 + np.exp(-z64))).max() < 1e-5
        zs, _ = o.triplet_scores(e, second, first, elbow)                     # swapped pair: a different input
        assert not np.array_equal(zs, z)
    za, _ = o.triplet_scores(e, first, second, False)
    ze, _ = o.triplet_scores(e, first, second, True)
    assert not np.array_equal(za, ze)                                        # two separate classifiers (L160)


def test_triplet_classifier_bf16_rounding_points():
    # R20 applied to the classifier: bf16 weights on the 2d -> d layer, hidden activation rounded, d -> 1 layer fp32
    cfg, W, blob = _triplet_model("bf16")
    lay = {n: (w, b) for n, w, b in W}
    rng = np.random.default_rng(5)
    e = torch_bf16(rng.normal(0, 1, (20, 16)).astype(F))                     # stored edge state: bf16 numbers
    first = rng.integers(0, 20, 40).astype(np.int32); second = rng.integers(0, 20, 40).astype(np.int32)
    z, _ = oracle.Oracle(blob, "bf16").triplet_scores(e, first, second, False)
    x = np.concatenate([e[first], e[second]], 1)
    hid = torch_bf16(np.maximum(f32_chain(x, torch_bf16(lay["tart0"][0]), lay["tart0"][1]), 0))
    ref = f32_chain(hid, *lay["tart1"])[:, 0]
    assert np.array_equal(z.view(np.uint32), ref.view(np.uint32))
    unrounded = f32_chain(np.maximum(f32_chain(x, torch_bf16(lay["tart0"][0]), lay["tart0"][1]), 0), *lay["tart1"])[:, 0]
    assert not np.array_equal(z, unrounded)


# ------------------------------------------------------------------ track building (sec. 5.4; R30, R31)
def _tracks_py(src, dst, keep, art, ka, left, kl, right, kr, min_hits):
    """The four phases written with sets and breadth-first searches (no union-find, no sorting of pairs)."""
    E = src.size
    kept = [i for i in range(E) if keep[i]]
    # (1) super-edges: connected components of the kept elbows
    adj = {i: set() for i in kept}
    for (f, s), k in ((left, kl), (right, kr)):
        for a, b, kk in zip(f, s, k):
            if kk:
                adj[int(a)].add(int(b)); adj[int(b)].add(int(a))
    sup = {}
    for i in kept:
        if i in sup:
            continue
        sup[i] = i; todo = [i]
        while todo:
            u = todo.pop()
            for v in adj[u]:
                if v not in sup:
                    sup[v] = i; todo.append(v)
    arts = {(sup[int(a)], sup[int(b)]) for a, b, kk in zip(art[0], art[1], ka) if kk and sup[int(a)] != sup[int(b)]}
    # (2) shared articulations
    succ, pred = {}, {}
    for x, y in arts:
        succ.setdefault(x, set()).add(y); pred.setdefault(y, set()).add(x)
    shared = {(x, y) for x, y in arts if len(succ[x]) >= 2 or len(pred[y]) >= 2}
    nodes = set(sup.values())
    nadj = {x: set() for x in nodes}
    for x, y in arts - shared:
        nadj[x].add(y); nadj[y].add(x)
    comp = {}
    for x in sorted(nodes):
        if x in comp:
            continue
        comp[x] = x; todo = [x]
        while todo:
            u = todo.pop()
            for v in nadj[u]:
                if v not in comp:
                    comp[v] = x; todo.append(v)
    # (3) tracks
    members = {}
    for i in kept:
        members.setdefault(comp[sup[i]], []).append(i)
    touched = set()
    sets = []
    for x, y in shared:
        touched |= {comp[x], comp[y]}
        sets.append({comp[x], comp[y]})
    sets += [{c} for c in set(comp.values()) if c not in touched]
    # (4) hits
    tracks = set()
    for cs in sets:
        hits = set()
        for c in cs:
            for e in members[c]:
                hits |= {int(src[e]), int(dst[e])}
        if len(hits) >= min_hits:
            tracks.add(tuple(sorted(hits)))
    return sorted(tracks)


def _as_lists(offs, hits):
    return [tuple(int(h) for h in hits[offs[t]:offs[t + 1]]) for t in range(offs.size - 1)]


@pytest.mark.parametrize("seed,min_hits", [(0, 3), (1, 3), (2, 2), (3, 4), (4, 3), (5, 1)])
def test_track_building_equals_an_independent_set_formulation(seed, min_hits):
    plane, src, dst, keep = _random_graph(seed, n=16, E=34)
    rng = np.random.default_rng(100 + seed)
    trip = {k: oracle.triplets(src, dst, keep, plane.size, k)[:2] for k in ("articulation", "left_elbow", "right_elbow")}
    ka = (rng.random(trip["articulation"][0].size) < 0.7).astype(np.uint8)
    kl = (rng.random(trip["left_elbow"][0].size) < 0.3).astype(np.uint8)
    kr = (rng.random(trip["right_elbow"][0].size) < 0.3).astype(np.uint8)
    offs, hits = oracle.tracks_from_triplets(src, dst, keep, trip["articulation"], ka, trip["left_elbow"], kl,
                                             trip["right_elbow"], kr, min_hits)
    got = _as_lists(offs, hits)
    want = _tracks_py(src, dst, keep, trip["articulation"], ka, trip["left_elbow"], kl, trip["right_elbow"], kr, min_hits)
    assert got == want
    assert len(got) > 0
    # invariants: lexicographic order without repeats (R31), ascending hits, every hit an end point of a kept edge
    assert got == sorted(set(got))
    ends = set(src[keep > 0].tolist()) | set(dst[keep > 0].tolist())
    for t in got:
        assert list(t) == sorted(set(t)) and len(t) >= min_hits and set(t) <= ends


def test_without_shared_articulations_tracks_are_the_components_of_the_edge_graph():
    # no elbow kept and every edge with at most one successor / predecessor: phases 2-4 reduce to a plain WCC of
    # the edge graph (L168), checked with scipy
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    src = np.array([0, 1, 2, 4, 5, 7], np.int32); dst = np.array([1, 2, 3, 5, 6, 8], np.int32)   # chains 0-1-2-3, 4-5-6, 7-8
    keep = np.ones(6, np.uint8)
    art = oracle.triplets(src, dst, keep, 9, "articulation")[:2]
    ka = np.ones(art[0].size, np.uint8)
    none = (np.zeros(0, np.int32), np.zeros(0, np.int32))
    offs, hits = oracle.tracks_from_triplets(src, dst, keep, art, ka, none, np.zeros(0, np.uint8), none, np.zeros(0, np.uint8), 2)
    ncomp, lab = connected_components(coo_matrix((np.ones(art[0].size), (art[0], art[1])), shape=(6, 6)), directed=False)
    want = sorted(tuple(sorted(set(src[lab == c].tolist()) | set(dst[lab == c].tolist()))) for c in range(ncomp))
    assert _as_lists(offs, hits) == want == [(0, 1, 2, 3), (4, 5, 6), (7, 8)]
    # a rejected articulation splits the chain (the triplet classifier separates tracks, L78)
    ka[0] = 0
    offs, hits = oracle.tracks_from_triplets(src, dst, keep, art, ka, none, np.zeros(0, np.uint8), none, np.zeros(0, np.uint8), 2)
    assert _as_lists(offs, hits) == [(0, 1), (1, 2, 3), (4, 5, 6), (7, 8)]


def test_electron_pair_sharing_its_first_hits_gives_two_tracks_with_the_shared_set_duplicated():
    # L168-170: an e+e- pair shares hits 0, 1 (edge 0 -> 1) and then separates: 1 -> 2 -> 4 and 1 -> 3 -> 5.
    # Both articulations out of the shared edge are genuine, the elbow (1 -> 2, 1 -> 3) is not (two particles).
    src = np.array([0, 1, 1, 2, 3], np.int32); dst = np.array([1, 2, 3, 4, 5], np.int32)
    keep = np.ones(5, np.uint8)
    art = oracle.triplets(src, dst, keep, 6, "articulation")[:2]
    left = oracle.triplets(src, dst, keep, 6, "left_elbow")[:2]
    right = oracle.triplets(src, dst, keep, 6, "right_elbow")[:2]
    assert list(zip(art[0].tolist(), art[1].tolist())) == [(0, 1), (0, 2), (1, 3), (2, 4)]
    assert list(zip(left[0].tolist(), left[1].tolist())) == [(1, 2)] and right[0].size == 0
    ka = np.ones(4, np.uint8)
    offs, hits = oracle.tracks_from_triplets(src, dst, keep, art, ka, left, np.zeros(1, np.uint8), right, np.zeros(0, np.uint8), 3)
    assert _as_lists(offs, hits) == [(0, 1, 2, 4), (0, 1, 3, 5)]                # hits 0, 1 in both tracks
    # a plain WCC on the purified hit graph (the paper's CUDA path, L206) merges the pair into one track
    tid = oracle.components(src, dst, np.ones(5, F), 0.0, 6)
    assert np.unique(tid).size == 1
    # if the elbow were accepted, 1 -> 2 and 1 -> 3 would be ONE super-edge with the two successors 2 -> 4 and 3 -> 5:
    # the sharing moves one step down and the merged set {0 -> 1, 1 -> 2, 1 -> 3} is what gets duplicated
    offs, hits = oracle.tracks_from_triplets(src, dst, keep, art, ka, left, np.ones(1, np.uint8), right, np.zeros(0, np.uint8), 3)
    assert _as_lists(offs, hits) == [(0, 1, 2, 3, 4), (0, 1, 2, 3, 5)]


def test_skipped_plane_elbows_remove_the_duplicate_articulations():
    # one particle, hits 0 .. 3 on consecutive planes, with the skip edge 0 -> 2 next to 0 -> 1, 1 -> 2 (window 2):
    # edge 2 -> 3 has two predecessors (1 -> 2 and 0 -> 2).  With the elbows accepted they are one super-edge and
    # the duplicate disappears ("duplicate edges resulting from elbow connections are removed"): one track.
    src = np.array([0, 0, 1, 2], np.int32); dst = np.array([1, 2, 2, 3], np.int32)
    keep = np.ones(4, np.uint8)
    art = oracle.triplets(src, dst, keep, 4, "articulation")[:2]
    left = oracle.triplets(src, dst, keep, 4, "left_elbow")[:2]
    right = oracle.triplets(src, dst, keep, 4, "right_elbow")[:2]
    assert list(zip(art[0].tolist(), art[1].tolist())) == [(0, 2), (1, 3), (2, 3)]
    assert list(zip(left[0].tolist(), left[1].tolist())) == [(0, 1)]
    assert list(zip(right[0].tolist(), right[1].tolist())) == [(1, 2)]
    ones = lambda t: np.ones(t[0].size, np.uint8)
    offs, hits = oracle.tracks_from_triplets(src, dst, keep, art, ones(art), left, ones(left), right, ones(right), 3)
    assert _as_lists(offs, hits) == [(0, 1, 2, 3)]
    # with the elbows rejected the same articulations are "shared" and the set is duplicated
    offs, hits = oracle.tracks_from_triplets(src, dst, keep, art, ones(art), left, np.zeros(1, np.uint8), right, np.zeros(1, np.uint8), 3)
    assert len(_as_lists(offs, hits)) == 2


def test_triplet_pipeline_on_a_noise_free_event_with_truth_scores():
    # truth edges of a noise-free event, every triplet of one particle accepted: every particle with >= 3 hits is
    # exactly one track (L78: triplets separate tracks; with perfect inputs nothing is shared)
    cfg = datagen.get_config("cfg0")
    b = datagen.generate_batch(cfg, n_events=2)
    src, dst, want = [], [], []
    for e in range(b.n_events):                                # particle ids are per event
        lo, hi = int(b.event_offsets[e]), int(b.event_offsets[e + 1])
        for pid in np.unique(b.particle[lo:hi]):
            idx = lo + np.nonzero(b.particle[lo:hi] == pid)[0]
            idx = idx[np.argsort(b.plane[idx], kind="stable")]
            assert np.all(np.diff(b.plane[idx]) > 0)
            src += idx[:-1].tolist(); dst += idx[1:].tolist()
            if idx.size >= 3:
                want.append(tuple(sorted(idx.tolist())))
    want.sort()
    order = np.lexsort((dst, src))
    src = np.asarray(src, np.int32)[order]; dst = np.asarray(dst, np.int32)[order]
    keep = np.ones(src.size, np.uint8)
    art = oracle.triplets(src, dst, keep, b.n_hits, "articulation")[:2]
    none = (np.zeros(0, np.int32), np.zeros(0, np.int32)); z8 = np.zeros(0, np.uint8)
    offs, hits = oracle.tracks_from_triplets(src, dst, keep, art, np.ones(art[0].size, np.uint8), none, z8, none, z8, 3)
    got = _as_lists(offs, hits)
    assert got == want and len(got) > 10


def test_run_triplets_end_to_end_shapes_and_thresholds():
    cfg = datagen.get_config("cfg0").replace(triplets=1)
    b = datagen.generate_batch(cfg)
    W = centred_parity_weights(cfg, b)
    o = oracle.Oracle(datagen.pack_blob(cfg, W), "fp32")
    r = o.run(b.xyz, b.plane, b.event_offsets, cfg.k, cfg.window)
    t = o.run_triplets(b.xyz, r["src"], r["dst"], cfg.threshold, cfg.triplet_threshold)
    assert np.array_equal(t["keep"] > 0, r["logit"] >= oracle.logit_threshold(cfg.threshold)) and 0 < t["keep"].sum() < t["keep"].size
    for kind in ("articulation", "left_elbow", "right_elbow"):
        assert t[kind]["first"].size > 0 and np.isfinite(t[kind]["logit"]).all()
    assert t["track_offsets"][0] == 0 and (np.diff(t["track_offsets"]) >= 3).all()
    # every hit of every track is a hit of the event; tracks may share hits (that is the point of sec. 5.4)
    assert t["track_hits"].max(initial=0) < b.n_hits


@pytest.mark.parametrize("seed", [0, 3, 5])
def test_components_then_tracks_equals_the_one_call_and_component_names_are_minimum_edge_ids(seed):
    plane, src, dst, keep = _random_graph(seed, n=16, E=34)
    rng = np.random.default_rng(200 + seed)
    trip = {k: oracle.triplets(src, dst, keep, plane.size, k)[:2] for k in ("articulation", "left_elbow", "right_elbow")}
    ka = (rng.random(trip["articulation"][0].size) < 0.7).astype(np.uint8)
    kl = (rng.random(trip["left_elbow"][0].size) < 0.3).astype(np.uint8)
    kr = (rng.random(trip["right_elbow"][0].size) < 0.3).astype(np.uint8)
    comp, shared = oracle.triplet_components(keep, trip["articulation"], ka, trip["left_elbow"], kl, trip["right_elbow"], kr)
    assert np.array_equal(comp >= 0, keep > 0)
    for c in np.unique(comp[comp >= 0]):
        assert c == np.flatnonzero(comp == c).min()              # a component is named by its smallest edge id
    assert shared.shape[0] > 0 and np.array_equal(shared, np.unique(shared, axis=0))
    assert set(shared.reshape(-1).tolist()) <= set(comp[comp >= 0].tolist())
    a = oracle.tracks_from_components(src, dst, comp, shared, 3)
    b = oracle.tracks_from_triplets(src, dst, keep, trip["articulation"], ka, trip["left_elbow"], kl, trip["right_elbow"], kr, 3)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
