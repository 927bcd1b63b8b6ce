"""ctypes binding of the CPU oracle (oracle/etx_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It shares nothing with the CUDA path
(paper_2407_12119_b200): neither imports the other.  Argument marshalling only; every
step of the method is in etx_oracle.cpp, where each function cites PAPER.md.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "etx_oracle.cpp")
_LIB = os.path.join(_HERE, "libetx_oracle.so")
# -ffp-contract=off: no silent fusion; fused multiply-adds are explicit std::fmaf (hardware FMA via -mfma).
_FLAGS = ["-O3", "-std=c++17", "-mavx2", "-mfma", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
          "-shared", "-fPIC"]
# ETX_ORACLE_SANITIZE=1: the same source under AddressSanitizer + UndefinedBehaviorSanitizer, as a library of its own
# (DESIGN.md sec. 5).  Python is not built with ASan, so its runtime has to be preloaded:
#   ETX_ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
#       python -m pytest tests/test_oracle_pins.py tests/test_oracle_triplets.py -q
if os.environ.get("ETX_ORACLE_SANITIZE") == "1":
    _LIB = os.path.join(_HERE, "libetx_oracle_san.so")
    _FLAGS = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] + _FLAGS[1:]

PRECISION = {"fp32": 0, "bf16": 1, "int8": 2}
STATE_DTYPE = {"auto": 0, "fp32": 1, "bf16": 2}     # storage of h, e, m; "bf16" only changes int8 mode (R21)


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", *_FLAGS, "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("n_planes", C.c_int32), ("norm_offset", C.c_float * 3), ("norm_div", C.c_float * 3),
                ("precision", C.c_int32), ("cyl_offset", C.c_float * 3), ("cyl_div", C.c_float * 3),
                ("state_dtype", C.c_int32)]


_lib = None


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.etxo_create.restype = C.c_void_p
        L.etxo_create.argtypes = [C.c_void_p, C.c_uint64, C.POINTER(_Params)]
        L.etxo_error.restype = C.c_char_p
        L.etxo_error.argtypes = [C.c_void_p]
        L.etxo_destroy.argtypes = [C.c_void_p]
        L.etxo_threads.restype = C.c_int
        L.etxo_set_threads.argtypes = [C.c_int]
        L.etxo_bf16_round.restype = C.c_float
        L.etxo_bf16_round.argtypes = [C.c_float]
        L.etxo_quant_i8.restype = C.c_int32
        L.etxo_quant_i8.argtypes = [C.c_float, C.c_float]
        L.etxo_record_absmax.argtypes = [C.c_void_p, C.c_int]
        L.etxo_n_layers.restype = C.c_int
        L.etxo_n_layers.argtypes = [C.c_void_p]
        L.etxo_get_absmax.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
        L.etxo_scales_from_absmax.restype = C.c_int
        L.etxo_scales_from_absmax.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
        L.etxo_set_tap.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32)]
        L.etxo_get_qweights.restype = C.c_int
        L.etxo_get_qweights.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int8), C.POINTER(C.c_float),
                                        C.POINTER(C.c_float)]
        L.etxo_plane_offsets.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_int, C.c_int,
                                         C.POINTER(C.c_int32)]
        L.etxo_features.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_float)]
        L.etxo_features_emb.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_float)]
        L.etxo_embed.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_float)]
        L.etxo_knn.argtypes = [C.POINTER(C.c_float), C.c_int64, C.c_int, C.POINTER(C.c_int32),
                               C.POINTER(C.c_int32), C.c_int, C.c_int, C.c_int, C.c_int, C.c_float,
                               C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.etxo_build_edges.restype = C.c_int64
        L.etxo_build_edges.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_int64, C.c_int,
                                       C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.etxo_csc.argtypes = [C.POINTER(C.c_int32), C.c_int64, C.c_int64, C.POINTER(C.c_int32),
                               C.POINTER(C.c_int32)]
        L.etxo_gnn.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_int32),
                               C.POINTER(C.c_int32), C.c_int64, C.POINTER(C.c_float), C.POINTER(C.c_float),
                               C.POINTER(C.c_float), C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_int]
        L.etxo_logit_threshold.restype = C.c_float
        L.etxo_logit_threshold.argtypes = [C.c_float]
        L.etxo_components.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_float),
                                      C.c_int64, C.c_float, C.c_int64, C.POINTER(C.c_int32)]
        L.etxo_tracks.restype = C.c_int64
        L.etxo_tracks.argtypes = [C.POINTER(C.c_int32), C.c_int64, C.POINTER(C.c_int32), C.c_int64, C.c_int32,
                                  C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        u8p = C.POINTER(C.c_uint8)
        L.etxo_triplets.restype = C.c_int64
        L.etxo_triplets.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_int32), u8p, C.c_int64, C.c_int64, C.c_int,
                                    C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.etxo_triplet_scores.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                          C.c_int64, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.etxo_has_triplets.restype = C.c_int
        L.etxo_has_triplets.argtypes = [C.c_void_p]
        L.etxo_tracks_from_triplets.restype = C.c_int64
        L.etxo_tracks_from_triplets.argtypes = ([C.POINTER(C.c_int32), C.POINTER(C.c_int32), u8p, C.c_int64]
                                                + [C.POINTER(C.c_int32), C.POINTER(C.c_int32), u8p, C.c_int64] * 3
                                                + [C.c_int32, C.POINTER(C.c_int32), C.c_int64, C.POINTER(C.c_int32), C.c_int64])
        L.etxo_triplet_components.restype = C.c_int64
        L.etxo_triplet_components.argtypes = ([u8p, C.c_int64] + [C.POINTER(C.c_int32), C.POINTER(C.c_int32), u8p, C.c_int64] * 3
                                              + [C.POINTER(C.c_int32)] * 3)
        L.etxo_tracks_from_components.restype = C.c_int64
        L.etxo_tracks_from_components.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_int64,
                                                  C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_int64, C.c_int32,
                                                  C.POINTER(C.c_int32), C.c_int64, C.POINTER(C.c_int32), C.c_int64]
        _lib = L
    return _lib


def threads() -> int:
    return int(lib().etxo_threads())


def set_threads(n: int) -> None:
    lib().etxo_set_threads(int(n))


def bf16_round(x: float) -> float:
    return float(lib().etxo_bf16_round(C.c_float(x)))


def quant_i8(x: float, scale: float) -> int:
    return int(lib().etxo_quant_i8(C.c_float(x), C.c_float(scale)))


def logit_threshold(thr: float) -> float:
    return float(lib().etxo_logit_threshold(C.c_float(thr)))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def plane_offsets(plane, event_offsets, n_planes=26):
    plane, eo = _i32(plane), _i32(event_offsets)
    B = eo.size - 1
    out = np.zeros(B * (n_planes + 1), np.int32)
    lib().etxo_plane_offsets(_p(plane, C.c_int32), _p(eo, C.c_int32), B, n_planes, _p(out, C.c_int32))
    return out.reshape(B, n_planes + 1)


def knn(emb, plane, event_offsets, k, window, d2_max=np.inf, n_planes=26):
    """-> (nbr [N,k] int32 (-1 padded), deg [N] int32)."""
    emb, plane, eo = _f32(emb), _i32(plane), _i32(event_offsets)
    n, nd = emb.shape if emb.ndim == 2 else (0, 4)
    nbr = np.full((n, k), -1, np.int32)
    deg = np.zeros(n, np.int32)
    lib().etxo_knn(_p(emb, C.c_float), n, nd, _p(plane, C.c_int32), _p(eo, C.c_int32), eo.size - 1,
                   n_planes, k, window, C.c_float(d2_max), _p(nbr, C.c_int32), _p(deg, C.c_int32))
    return nbr, deg


def build_edges(nbr, deg):
    """-> (src [E], dst [E], row_ptr [N+1])."""
    nbr, deg = _i32(nbr), _i32(deg)
    n, k = nbr.shape
    cap = max(int(deg.sum()), 1)
    src, dst = np.zeros(cap, np.int32), np.zeros(cap, np.int32)
    row_ptr = np.zeros(n + 1, np.int32)
    E = lib().etxo_build_edges(_p(nbr, C.c_int32), _p(deg, C.c_int32), n, k, _p(src, C.c_int32),
                               _p(dst, C.c_int32), _p(row_ptr, C.c_int32))
    return src[:E].copy(), dst[:E].copy(), row_ptr


def csc(dst, n):
    dst = _i32(dst)
    col_ptr = np.zeros(n + 1, np.int32)
    in_edge = np.zeros(max(dst.size, 1), np.int32)
    lib().etxo_csc(_p(dst, C.c_int32), dst.size, n, _p(col_ptr, C.c_int32), _p(in_edge, C.c_int32))
    return col_ptr, in_edge[:dst.size].copy()


def components(src, dst, logit, tau, n):
    src, dst, logit = _i32(src), _i32(dst), _f32(logit)
    out = np.zeros(n, np.int32)
    lib().etxo_components(_p(src, C.c_int32), _p(dst, C.c_int32), _p(logit, C.c_float), src.size,
                          C.c_float(tau), n, _p(out, C.c_int32))
    return out


def tracks(track_id, event_offsets, min_hits=3):
    """Track containers from the per-hit component labels (etxo_tracks)."""
    tid, eo = _i32(track_id), _i32(event_offsets)
    n, B = tid.size, eo.size - 1
    index = np.zeros(n, np.int32); offs = np.zeros(n + 1, np.int32); hits = np.zeros(max(n, 1), np.int32)
    ev = np.zeros(B + 1, np.int32)
    T = int(lib().etxo_tracks(_p(tid, C.c_int32), n, _p(eo, C.c_int32), B, int(min_hits), _p(index, C.c_int32),
                              _p(offs, C.c_int32), _p(hits, C.c_int32), _p(ev, C.c_int32)))
    return dict(n_tracks=T, track_index=index, track_offsets=offs[:T + 1].copy(), track_hits=hits[:offs[T]].copy(),
                event_track_offsets=ev)


TRIPLET_KINDS = {"articulation": 0, "left_elbow": 1, "right_elbow": 2}


def _u8(a):
    return np.ascontiguousarray(a, dtype=np.uint8)


def triplets(src, dst, keep, n, kind):
    """Triplets of one kind on the purified hit graph (etxo_triplets).  -> (first [T], second [T], hit [T])."""
    src, dst, keep = _i32(src), _i32(dst), _u8(keep)
    k = TRIPLET_KINDS[kind] if isinstance(kind, str) else int(kind)
    null = C.POINTER(C.c_int32)()
    T = int(lib().etxo_triplets(_p(src, C.c_int32), _p(dst, C.c_int32), _p(keep, C.c_uint8), src.size, n, k, null, null, null))
    a, b, h = (np.zeros(max(T, 1), np.int32) for _ in range(3))
    lib().etxo_triplets(_p(src, C.c_int32), _p(dst, C.c_int32), _p(keep, C.c_uint8), src.size, n, k,
                        _p(a, C.c_int32), _p(b, C.c_int32), _p(h, C.c_int32))
    return a[:T].copy(), b[:T].copy(), h[:T].copy()


def tracks_from_triplets(src, dst, keep, art, keep_art, left, keep_left, right, keep_right, min_hits=3):
    """The four phases of PAPER.md sec. 5.4 (etxo_tracks_from_triplets).  art / left / right = (first, second) edge-id
    arrays, keep_* their kept flags.  -> (track_offsets [T + 1], track_hits)."""
    src, dst, keep = _i32(src), _i32(dst), _u8(keep)
    E = src.size
    args = []
    n_shared_max = 0
    for (f, s), kf in ((art, keep_art), (left, keep_left), (right, keep_right)):
        f, s, kf = _i32(f), _i32(s), _u8(kf)
        args += [f, s, kf]
        n_shared_max = max(n_shared_max, f.size)
    cap_tracks = E + int(np.asarray(art[0]).size) + 1
    cap_hits = 2 * (E + 1) * 2 + 4 * int(np.asarray(art[0]).size) * 64 + 16
    while True:
        offs = np.zeros(cap_tracks + 1, np.int32); hits = np.zeros(cap_hits, np.int32)
        T = int(lib().etxo_tracks_from_triplets(
            _p(src, C.c_int32), _p(dst, C.c_int32), _p(keep, C.c_uint8), E,
            _p(args[0], C.c_int32), _p(args[1], C.c_int32), _p(args[2], C.c_uint8), args[0].size,
            _p(args[3], C.c_int32), _p(args[4], C.c_int32), _p(args[5], C.c_uint8), args[3].size,
            _p(args[6], C.c_int32), _p(args[7], C.c_int32), _p(args[8], C.c_uint8), args[6].size,
            int(min_hits), _p(offs, C.c_int32), cap_tracks, _p(hits, C.c_int32), cap_hits))
        if T >= 0:
            return offs[:T + 1].copy(), hits[:offs[T]].copy()
        cap_hits *= 4


def triplet_components(keep, art, keep_art, left, keep_left, right, keep_right):
    """Phases (1)-(2) of sec. 5.4 (etxo_triplet_components).  -> (edge_comp [E], shared [n, 2] sorted, unique)."""
    keep = _u8(keep)
    E = keep.size
    args = []
    for (f, s), kf in ((art, keep_art), (left, keep_left), (right, keep_right)):
        args += [_i32(f), _i32(s), _u8(kf)]
    TA = args[0].size
    comp = np.zeros(max(E, 1), np.int32); sx = np.zeros(max(TA, 1), np.int32); sy = np.zeros(max(TA, 1), np.int32)
    n = int(lib().etxo_triplet_components(
        _p(keep, C.c_uint8), E,
        _p(args[0], C.c_int32), _p(args[1], C.c_int32), _p(args[2], C.c_uint8), args[0].size,
        _p(args[3], C.c_int32), _p(args[4], C.c_int32), _p(args[5], C.c_uint8), args[3].size,
        _p(args[6], C.c_int32), _p(args[7], C.c_int32), _p(args[8], C.c_uint8), args[6].size,
        _p(comp, C.c_int32), _p(sx, C.c_int32), _p(sy, C.c_int32)))
    return comp[:E].copy(), np.stack([sx[:n], sy[:n]], axis=1).astype(np.int32)


def tracks_from_components(src, dst, edge_comp, shared, min_hits=3):
    """Phases (3)-(4) of sec. 5.4 (etxo_tracks_from_components).  -> (track_offsets [T + 1], track_hits)."""
    src, dst, comp = _i32(src), _i32(dst), _i32(edge_comp)
    shared = np.asarray(shared, np.int32).reshape(-1, 2)
    sx, sy = _i32(shared[:, 0]), _i32(shared[:, 1])
    E = src.size
    cap_tracks = E + shared.shape[0] + 1
    cap_hits = 4 * (E + 1) + 16
    while True:
        offs = np.zeros(cap_tracks + 1, np.int32); hits = np.zeros(cap_hits, np.int32)
        T = int(lib().etxo_tracks_from_components(_p(src, C.c_int32), _p(dst, C.c_int32), _p(comp, C.c_int32), E,
                                                  _p(sx, C.c_int32), _p(sy, C.c_int32), shared.shape[0], int(min_hits),
                                                  _p(offs, C.c_int32), cap_tracks, _p(hits, C.c_int32), cap_hits))
        if T >= 0:
            return offs[:T + 1].copy(), hits[:offs[T]].copy()
        cap_hits *= 4


class Oracle:
    """One model (weights blob + precision mode).  Methods mirror the stages of the hot path."""

    def __init__(self, blob: bytes, precision: str = "fp32", n_planes: int = 26,
                 norm_offset=(0.0, 0.0, 300.0), norm_div=(40.0, 40.0, 1050.0),
                 cyl_offset=(-20.0, 0.0, 300.0), cyl_div=(12.0, 3.14159274, 1050.0), state_dtype: str = "auto"):
        prm = _Params(n_planes, (C.c_float * 3)(*norm_offset), (C.c_float * 3)(*norm_div),
                      PRECISION[precision], (C.c_float * 3)(*cyl_offset), (C.c_float * 3)(*cyl_div),
                      STATE_DTYPE[state_dtype])
        self._blob = bytes(blob)
        self._h = lib().etxo_create(self._blob, len(self._blob), C.byref(prm))
        err = lib().etxo_error(self._h).decode()
        if err:
            lib().etxo_destroy(self._h)
            self._h = None
            raise ValueError("oracle: " + err)
        self.n_planes = n_planes
        self.precision = precision
        import struct
        hdr = struct.unpack("<16I", self._blob[:64])
        self.emb_dim, self.latent = hdr[4], hdr[5]
        self.emb_input = hdr[10]          # 0: Cartesian features, 1: cylindrical (R27)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().etxo_destroy(self._h)
            self._h = None

    def features(self, xyz):
        xyz = _f32(xyz)
        out = np.zeros_like(xyz)
        lib().etxo_features(self._h, _p(xyz, C.c_float), xyz.shape[0], _p(out, C.c_float))
        return out

    def features_emb(self, xyz):
        """Input of the embedding MLP (the Cartesian features, or normalised (r, phi, z) when the blob says so)."""
        xyz = _f32(xyz)
        out = np.zeros_like(xyz)
        lib().etxo_features_emb(self._h, _p(xyz, C.c_float), xyz.shape[0], _p(out, C.c_float))
        return out

    def embed(self, xyz):
        xyz = _f32(xyz)
        out = np.zeros((xyz.shape[0], self.emb_dim), np.float32)
        lib().etxo_embed(self._h, _p(xyz, C.c_float), xyz.shape[0], _p(out, C.c_float))
        return out

    def gnn(self, xyz, src, dst, want_states=False, m_iter=-1):
        """-> dict(logit, score[, h, e, m])."""
        xyz, src, dst = _f32(xyz), _i32(src), _i32(dst)
        n, E, d = xyz.shape[0], src.size, self.latent
        logit, score = np.zeros(E, np.float32), np.zeros(E, np.float32)
        h = np.zeros((n, d), np.float32) if want_states else None
        e = np.zeros((E, d), np.float32) if want_states else None
        m = np.zeros((n, 2 * d), np.float32) if m_iter >= 0 else None
        null = C.POINTER(C.c_float)()
        lib().etxo_gnn(self._h, _p(xyz, C.c_float), n, _p(src, C.c_int32), _p(dst, C.c_int32), E,
                       _p(logit, C.c_float), _p(score, C.c_float),
                       _p(h, C.c_float) if h is not None else null,
                       _p(e, C.c_float) if e is not None else null,
                       _p(m, C.c_float) if m is not None else null, m_iter)
        out = {"logit": logit, "score": score}
        if want_states:
            out["h"], out["e"] = h, e
        if m is not None:
            out["m"] = m
        return out

    def has_triplets(self) -> bool:
        return bool(lib().etxo_has_triplets(self._h))

    def triplet_scores(self, e_state, first, second, elbow: bool):
        """Triplet classifier on pairs of final edge encodings (etxo_triplet_scores).  -> (logit [T], score [T])."""
        e_state, first, second = _f32(e_state), _i32(first), _i32(second)
        T = first.size
        logit, score = np.zeros(max(T, 1), np.float32), np.zeros(max(T, 1), np.float32)
        lib().etxo_triplet_scores(self._h, _p(e_state, C.c_float), _p(first, C.c_int32), _p(second, C.c_int32), T,
                                  int(bool(elbow)), _p(logit, C.c_float), _p(score, C.c_float))
        return logit[:T].copy(), score[:T].copy()

    def run_triplets(self, xyz, src, dst, threshold=0.5, triplet_threshold=0.5, min_hits=3):
        """Steps 4-7 of Figure 3 (L94) on a given rough graph: edge scores, purified hit graph, triplets of the
        three kinds, their scores, purified edge graph, tracks.  -> dict."""
        g = self.gnn(xyz, src, dst, want_states=True)
        keep = (g["logit"] >= logit_threshold(threshold)).astype(np.uint8)
        tau_t = logit_threshold(triplet_threshold)
        n = np.asarray(xyz).shape[0]
        out = dict(logit=g["logit"], keep=keep, e=g["e"])
        kept = {}
        for kind in ("articulation", "left_elbow", "right_elbow"):
            f, s, h = triplets(src, dst, keep, n, kind)
            z, sc = self.triplet_scores(g["e"], f, s, elbow=(kind != "articulation"))
            out[kind] = dict(first=f, second=s, hit=h, logit=z, score=sc)
            kept[kind] = (z >= tau_t).astype(np.uint8)
        offs, hits = tracks_from_triplets(src, dst, keep,
                                          (out["articulation"]["first"], out["articulation"]["second"]), kept["articulation"],
                                          (out["left_elbow"]["first"], out["left_elbow"]["second"]), kept["left_elbow"],
                                          (out["right_elbow"]["first"], out["right_elbow"]["second"]), kept["right_elbow"],
                                          min_hits)
        out["track_offsets"], out["track_hits"] = offs, hits
        return out

    # --- instrumentation ---------------------------------------------------------------
    def n_layers(self) -> int:
        return int(lib().etxo_n_layers(self._h))

    def record_absmax(self, on: bool):
        lib().etxo_record_absmax(self._h, int(on))

    def absmax(self):
        out = np.zeros(self.n_layers(), np.float32)
        lib().etxo_get_absmax(self._h, _p(out, C.c_float))
        return out

    def scales_from_absmax(self):
        out = np.zeros(self.n_layers(), np.float32)
        n = lib().etxo_scales_from_absmax(self._h, _p(out, C.c_float))
        return out[:n].copy()

    def set_tap(self, layer_index: int, out: np.ndarray | None):
        """int8 mode: copy the int32 accumulators of layer `layer_index` (blob order) into `out` [rows, out]."""
        self._tap = out
        lib().etxo_set_tap(self._h, layer_index if out is not None else -1,
                           _p(out, C.c_int32) if out is not None else C.POINTER(C.c_int32)())

    def qweights(self, layer_index: int, out_dim: int, in_dim: int):
        Wq = np.zeros((out_dim, in_dim), np.int8)
        sw = np.zeros(out_dim, np.float32)
        sx = C.c_float(0)
        ok = lib().etxo_get_qweights(self._h, layer_index, _p(Wq, C.c_int8), _p(sw, C.c_float), C.byref(sx))
        return (Wq, sw, float(sx.value)) if ok else None

    # --- the whole path ----------------------------------------------------------------
    def run(self, xyz, plane, event_offsets, k, window, d2_max=np.inf, threshold=0.5):
        """All five stages.  -> dict(emb, nbr, deg, src, dst, row_ptr, logit, score, track_id)."""
        emb = self.embed(xyz)
        nbr, deg = knn(emb, plane, event_offsets, k, window, d2_max, self.n_planes)
        src, dst, row_ptr = build_edges(nbr, deg)
        g = self.gnn(xyz, src, dst)
        tid = components(src, dst, g["logit"], logit_threshold(threshold), np.asarray(xyz).shape[0])
        return dict(emb=emb, nbr=nbr, deg=deg, src=src, dst=dst, row_ptr=row_ptr,
                    logit=g["logit"], score=g["score"], track_id=tid)


def calibrate_int8(blob_fp32: bytes, xyz, plane, event_offsets, k, window, d2_max=np.inf, threshold=0.5) -> np.ndarray:
    """Activation scales s_x = max|x|/127 per quantised Linear from the fp32 forward on a
    calibration batch (reading R21).  -> fp32 array in blob order."""
    o = Oracle(blob_fp32, "fp32")
    o.record_absmax(True)
    emb = o.embed(xyz)
    nbr, deg = knn(emb, plane, event_offsets, k, window, d2_max)
    src, dst, _ = build_edges(nbr, deg)
    if o.has_triplets():
        o.run_triplets(xyz, src, dst, threshold, threshold)
    else:
        o.gnn(xyz, src, dst)
    o.record_absmax(False)
    return o.scales_from_absmax()


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
