"""Independent checkers used to pin the oracle (and later the CUDA path).  None of this is
imported by the oracle or by the product; each checker is a different formulation from the
oracle's (brute force, exact rationals, dense matrices, BFS, the paper's sweeps)."""
from __future__ import annotations

from fractions import Fraction

import numpy as np

import datagen
from datagen.configs import EtxConfig


def toy_config(d=2, L=1, D=4, H=1, k=4, w=1, edge_enc_input=0, precision="fp32") -> EtxConfig:
    return datagen.get_config("cfg0").replace(name="toy", emb_hidden=D, emb_n_hidden_layers=H, gnn_latent=d,
                                              gnn_iters=L, k=k, window=w, edge_enc_input=edge_enc_input,
                                              precision=precision)


def zero_layers(cfg):
    return [(n, np.zeros((o, i), np.float32), np.zeros(o, np.float32)) for (n, o, i) in datagen.layer_shapes(cfg)]


def set_layer(layers, name, W=None, b=None):
    for idx, (n, W0, b0) in enumerate(layers):
        if n == name:
            layers[idx] = (n, np.asarray(W if W is not None else W0, np.float32).reshape(W0.shape),
                           np.asarray(b if b is not None else b0, np.float32).reshape(b0.shape))
            return
    raise KeyError(name)


# ---- exact fp32 arithmetic by rationals -------------------------------------------------
def round_f32(q: Fraction) -> np.float32:
    """Round an exact rational to the nearest fp32, ties to even (normal range only)."""
    if q == 0:
        return np.float32(0.0)
    s = -1 if q < 0 else 1
    q = abs(q)
    e = 0
    while q >= 2:
        q /= 2; e += 1
    while q < 1:
        q *= 2; e -= 1
    m = q * (1 << 23)                      # in [2^23, 2^24)
    fl = m.numerator // m.denominator
    rem = m - fl
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (fl & 1)):
        fl += 1
    assert -126 <= e <= 127, "subnormal/overflow not handled in this checker"
    return np.float32(s * float(Fraction(fl) * Fraction(2) ** (e - 23)))


def d2_exact_f32(a, b) -> np.float32:
    """Eq.(1) in the pinned order: t0*t0, then fma(t_i, t_i, d2), each step one fp32 rounding."""
    a = np.asarray(a, np.float32); b = np.asarray(b, np.float32)
    t = np.float32(a[0] - b[0])
    d2 = round_f32(Fraction(float(t)) * Fraction(float(t)))
    for i in range(1, a.size):
        t = np.float32(a[i] - b[i])
        d2 = round_f32(Fraction(float(t)) * Fraction(float(t)) + Fraction(float(d2)))
    return d2


def knn_bruteforce(emb, plane, event_offsets, k, w, d2_max=np.inf, n_planes=26):
    """All pairs of the event, filtered by plane window, full sort by (d2, index)."""
    n = emb.shape[0]
    nbr = np.full((n, k), -1, np.int32)
    deg = np.zeros(n, np.int32)
    for e in range(len(event_offsets) - 1):
        lo, hi = int(event_offsets[e]), int(event_offsets[e + 1])
        for q in range(lo, hi):
            cand = []
            for c in range(lo, hi):
                dp = int(plane[c]) - int(plane[q])
                if 1 <= dp <= w:
                    d2 = d2_exact_f32(emb[q], emb[c])
                    if d2 < d2_max:
                        cand.append((float(d2), c))
            cand.sort()
            cand = cand[:k]
            deg[q] = len(cand)
            for s, (_, c) in enumerate(cand):
                nbr[q, s] = c
    return nbr, deg


def knn_replace_the_max(emb, plane, event_offsets, k, w, d2_max=np.inf):
    """The paper's own loop (sec. 7.2): scan candidates, fill k slots, then replace
    the current maximum when a closer candidate comes.  Returns neighbour SETS per hit."""
    out = []
    for e in range(len(event_offsets) - 1):
        lo, hi = int(event_offsets[e]), int(event_offsets[e + 1])
        for q in range(lo, hi):
            slots = []
            for c in range(lo, hi):
                dp = int(plane[c]) - int(plane[q])
                if not (1 <= dp <= w):
                    continue
                d2 = float(d2_exact_f32(emb[q], emb[c]))
                if not d2 < d2_max:
                    continue
                if len(slots) < k:
                    slots.append((d2, c))
                else:
                    im = max(range(k), key=lambda s: slots[s][0])
                    if d2 < slots[im][0]:
                        slots[im] = (d2, c)
            out.append(set(c for _, c in slots))
    return out


# ---- components ------------------------------------------------------------------------
def components_bfs(src, dst, keep, n):
    adj = [[] for _ in range(n)]
    for s, t, kk in zip(src, dst, keep):
        if kk:
            adj[s].append(t); adj[t].append(s)
    lab = np.full(n, -1, np.int32)
    for r in range(n):                       # ascending: r is the min index of its component
        if lab[r] >= 0:
            continue
        lab[r] = r
        stack = [r]
        while stack:
            u = stack.pop()
            for v in adj[u]:
                if lab[v] < 0:
                    lab[v] = r; stack.append(v)
    return lab


def components_paper_sweeps(src, dst, keep, plane, n, n_planes=26, max_rounds=1000, stop_after=None):
    """PAPER.md L261 sec. 7.3: label = own index; forward sweep over planes taking the lowest label
    among left neighbours, then backward sweep over right neighbours; iterated to a fixed point.
    Returns (labels, rounds), rounds = the number of forward + backward rounds that still changed a
    label, plus the final one that changed nothing.  stop_after = r returns the labels after exactly r
    rounds (the paper's own algorithm is stop_after = 1)."""
    lab = np.arange(n, dtype=np.int64)
    left = [[] for _ in range(n)]; right = [[] for _ in range(n)]
    for s, t, kk in zip(src, dst, keep):
        if kk:
            right[s].append(t); left[t].append(s)
    by_plane = [np.nonzero(plane == p)[0] for p in range(n_planes)]
    for rnd in range(1, max_rounds + 1):
        changed = False
        for p in range(n_planes):
            for v in by_plane[p]:
                for u in left[v]:
                    if lab[u] < lab[v]:
                        lab[v] = lab[u]; changed = True
        for p in range(n_planes - 1, -1, -1):
            for v in by_plane[p]:
                for u in right[v]:
                    if lab[u] < lab[v]:
                        lab[v] = lab[u]; changed = True
        if not changed or (stop_after is not None and rnd >= stop_after):
            return lab.astype(np.int32), rnd
    raise RuntimeError("sweeps did not converge")


def check_edge_invariants(src, dst, row_ptr, plane, event_offsets, k, w):
    """PAPER.md L76/L101/L137: same event, plane[dst]-plane[src] in [1,w], out-degree <= k, no duplicates,
    src ascending, row_ptr = prefix sums."""
    n = plane.size
    ev = np.repeat(np.arange(len(event_offsets) - 1), np.diff(event_offsets))
    assert np.all(ev[src] == ev[dst])
    dp = plane[dst].astype(np.int64) - plane[src]
    assert np.all((dp >= 1) & (dp <= w))
    deg = np.bincount(src, minlength=n)
    assert deg.max(initial=0) <= k
    assert np.all(np.diff(src) >= 0)
    assert np.array_equal(row_ptr, np.concatenate([[0], np.cumsum(deg)]).astype(np.int32))
    key = src.astype(np.int64) * n + dst
    assert np.unique(key).size == key.size


def check_track_invariants(tid, src, dst, keep, event_offsets):
    n = tid.size
    idx = np.arange(n)
    assert np.all(tid <= idx)
    assert np.array_equal(tid[tid], tid)
    assert np.all(tid[src[keep]] == tid[dst[keep]])
    ev = np.repeat(np.arange(len(event_offsets) - 1), np.diff(event_offsets))
    assert np.all(ev[tid] == ev)


def centred_parity_weights(cfg, batch, seed=None):
    """"parity" preset weights with the head bias moved to -median(logit) of `batch` (computed with the
    fp32 oracle), so that scores spread around 0.5 and the threshold keeps about half of the edges
    (SURVEY.md sec. 8(c) A24).  Test utility: the product never sees how the bias was chosen."""
    import oracle
    layers = datagen.make_weights(cfg, "parity", seed=seed)
    o = oracle.Oracle(datagen.pack_blob(cfg, layers), "fp32")
    r = o.run(batch.xyz, batch.plane, batch.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    med = float(np.median(r["logit"])) if r["logit"].size else 0.0
    names = [l[0] for l in layers]
    ih = names.index("head")
    name, W, b = layers[ih]
    layers[ih] = (name, W, (b - np.float32(med)).astype(np.float32))
    if getattr(cfg, "triplets", 0):
        # the triplet classifiers likewise: biases moved so that about half of the triplets of each kind are kept
        o = oracle.Oracle(datagen.pack_blob(cfg, layers), "fp32")
        t = o.run_triplets(batch.xyz, r["src"], r["dst"], cfg.threshold, cfg.triplet_threshold)
        za = t["articulation"]["logit"]
        ze = np.concatenate([t["left_elbow"]["logit"], t["right_elbow"]["logit"]])
        for lname, z in (("tart1", za), ("telb1", ze)):
            i = names.index(lname)
            name, W, b = layers[i]
            layers[i] = (name, W, (b - np.float32(np.median(z) if z.size else 0.0)).astype(np.float32))
    return layers


# ---- the interaction network restated with explicit rounding points ------------------------
def f32_chain(x, W, b):
    """One Linear in the pinned fp32 order (R3): acc = 0; acc = fma(x[j], W[c][j], acc) for j
    ascending; y = acc + b[c].  Each fma is emulated as an exact float64 product and sum rounded once to
    fp32 (a 24 x 24 bit product is exact in float64)."""
    x = np.asarray(x, np.float32); W = np.asarray(W, np.float32); b = np.asarray(b, np.float32)
    acc = np.zeros((x.shape[0], W.shape[0]), np.float32)
    for j in range(W.shape[1]):
        acc = (x[:, j:j + 1].astype(np.float64) * W[None, :, j].astype(np.float64) + acc.astype(np.float64)).astype(np.float32)
    return (acc + b[None, :]).astype(np.float32)


def torch_bf16(x):
    """RNE rounding to bfloat16 by torch's CPU conversion (not the oracle's bit manipulation)."""
    import torch
    return torch.from_numpy(np.ascontiguousarray(x, np.float32)).to(torch.bfloat16).to(torch.float32).numpy()


BF16_POINTS = ("weights", "enc_hidden", "enc_out", "msg", "node_hidden", "h_resid", "edge_hidden", "e_resid")


def gnn_restated(cfg, layers, f, src, dst, points=(), on_linear_input=None):
    """PAPER.md L133-142 (sec. 5.2) written out with numpy, one statement per step of the paper, every
    Linear in the pinned fp32 order.  `points` names the places where a value is rounded to bfloat16
    (R20): "weights" (Linears with K >= 16 except the head), hidden activations of the four
    MLP kinds, encoder outputs, the message after its fp32 sum, h / e after the fp32 residual add.
    `on_linear_input(name, x)` sees the input tensor of every Linear (used to recompute INT8 scales).
    -> dict(h, e, logit)."""
    lay = {n: (W.astype(np.float32), b.astype(np.float32)) for n, W, b in layers}
    rnd = lambda x, p: torch_bf16(x) if p in points else x

    def linear(name, x):
        W, b = lay[name]
        if on_linear_input is not None:
            on_linear_input(name, x)
        if W.shape[1] >= 16 and name != "head" and "weights" in points:
            W = torch_bf16(W)
        return f32_chain(x, W, b)

    def mlp(n0, n1, x, hidden_point):
        a = rnd(np.maximum(linear(n0, x), np.float32(0)), hidden_point)
        return linear(n1, a)

    f = np.asarray(f, np.float32)
    n, E, d = f.shape[0], src.size, cfg.gnn_latent
    h = rnd(mlp("nenc0", "nenc1", f, "enc_hidden"), "enc_out")                        # L133
    x = np.abs(f[dst] - f[src]) if cfg.edge_enc_input == 0 else np.concatenate([h[src], h[dst]], 1)
    e = rnd(mlp("eenc0", "eenc1", x, "enc_hidden"), "enc_out")
    for it in range(cfg.gnn_iters):                                                   # L135-140
        m = np.zeros((n, 2 * d), np.float32)
        for i in range(E):                                                            # Eq.(4), ascending edge id
            m[src[i], :d] = m[src[i], :d] + e[i]
            m[dst[i], d:] = m[dst[i], d:] + e[i]
        m = rnd(m, "msg")
        h = rnd((h + mlp(f"node{it}_0", f"node{it}_1", np.concatenate([h, m], 1), "node_hidden")).astype(np.float32), "h_resid")
        e = rnd((e + mlp(f"edge{it}_0", f"edge{it}_1", np.concatenate([h[src], h[dst], e], 1), "edge_hidden")).astype(np.float32), "e_resid")
    logit = linear("head", e)[:, 0]                                                   # L142
    return dict(h=h, e=e, logit=logit)


def embed_restated(cfg, layers, f_emb, on_linear_input=None):
    """PAPER.md L96 (sec. 5.1): the embedding MLP in the pinned fp32 order, ReLU after hidden layers."""
    lay = {n: (W.astype(np.float32), b.astype(np.float32)) for n, W, b in layers}
    a = np.asarray(f_emb, np.float32)
    H = cfg.emb_n_hidden_layers
    for l in range(H + 1):
        if on_linear_input is not None:
            on_linear_input(f"emb{l}", a)
        a = f32_chain(a, *lay[f"emb{l}"])
        if l < H:
            a = np.maximum(a, np.float32(0))
    return a


def gnn_restated_int8(cfg, layers, scales, f, src, dst, state_bf16):
    """PAPER.md L133-142 in INT8 mode (R21) written out with numpy: every Linear with K >= 16 except the
    head quantises its input tensor (q = clamp(rne(x * (1 / s_x)), +-127), one fp32 multiply), multiplies integer
    codes (int64 matmul) and dequantises with y = fma((float) acc, s_x * s_w[c], b[c]); the K = 3 layers and the head
    are the pinned fp32 chain.  state_bf16: h, e and the message are rounded to bfloat16 (torch) when stored.
    -> dict(h, e, logit)."""
    F = np.float32
    lay = {n: (W.astype(F), b.astype(F)) for n, W, b in layers}
    qnames = [n for n, W, b in layers if W.shape[1] >= 16 and n not in ("head", "tart1", "telb1")]
    sx = {n: F(s) for n, s in zip(qnames, scales)}
    st = (lambda x: torch_bf16(x)) if state_bf16 else (lambda x: x)

    def linear(name, x):
        W, b = lay[name]
        if name not in sx:
            return f32_chain(x, W, b)
        inv = F(1.0) / sx[name]
        q = np.clip(np.rint((x.astype(F) * inv).astype(F)), -127, 127).astype(np.int64)
        amax = np.abs(W).max(1)
        sw = np.where(amax > 0, (amax / F(127)).astype(F), F(1.0)).astype(F)
        Wq = np.clip(np.rint((W / sw[:, None]).astype(F)), -127, 127).astype(np.int64)
        acc = q @ Wq.T
        scale = (sx[name] * sw).astype(F)
        return (acc.astype(np.float64) * scale.astype(np.float64)[None, :] + b.astype(np.float64)[None, :]).astype(F)

    mlp = lambda n0, n1, x: linear(n1, np.maximum(linear(n0, x), F(0)))
    f = np.asarray(f, F)
    n, E, d = f.shape[0], src.size, cfg.gnn_latent
    h = st(mlp("nenc0", "nenc1", f))
    x = np.abs(f[dst] - f[src]) if cfg.edge_enc_input == 0 else np.concatenate([h[src], h[dst]], 1)
    e = st(mlp("eenc0", "eenc1", x))
    for it in range(cfg.gnn_iters):
        m = np.zeros((n, 2 * d), F)
        for i in range(E):
            m[src[i], :d] = m[src[i], :d] + e[i]
            m[dst[i], d:] = m[dst[i], d:] + e[i]
        m = st(m)
        h = st((h + mlp(f"node{it}_0", f"node{it}_1", np.concatenate([h, m], 1))).astype(F))
        e = st((e + mlp(f"edge{it}_0", f"edge{it}_1", np.concatenate([h[src], h[dst], e], 1))).astype(F))
    logit = f32_chain(e, *lay["head"])[:, 0]
    return dict(h=h, e=e, logit=logit)
