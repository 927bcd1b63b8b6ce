"""ctypes binding of include/etx.h.  Marshalling only."""
from __future__ import annotations

import ctypes as C
import math
import os
import re

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libetx.so")
_HEADER = os.path.join(HERE, "..", "include", "etx.h")

PRECISION = {"fp32": 0, "bf16": 1, "int8": 2}
ENGINE = {"auto": 0, "simt": 1, "tc_serial": 2}
STATE_DTYPE = {"auto": 0, "fp32": 1, "bf16": 2}
STAGE_NAMES = ["S0_plane_offsets", "S1_embedding", "S2_knn", "S3_compaction_csc", "S4_encoders",
               "S4c_scatter", "S4d_node_net", "S4e_edge_net_head", "S5_components"]
STATUS = {0: "ETX_OK", -1: "ETX_ERR_ARG", -2: "ETX_ERR_BLOB", -3: "ETX_ERR_CAPACITY", -4: "ETX_ERR_INPUT_ORDER",
          -5: "ETX_ERR_CUDA", -6: "ETX_ERR_UNSUPPORTED"}


class EtxError(RuntimeError):
    def __init__(self, status: int, msg: str = ""):
        self.status = status
        super().__init__(f"{STATUS.get(status, status)}: {msg}")


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)      # optional device allocator callbacks (include/etx.h)
DEALLOC_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Hyperparams(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_planes", C.c_int32), ("norm_offset", C.c_float * 3),
                ("norm_div", C.c_float * 3), ("emb_hidden", C.c_int32), ("emb_n_hidden_layers", C.c_int32),
                ("emb_dim", C.c_int32), ("k", C.c_int32), ("window", C.c_int32), ("d2_max", C.c_float),
                ("gnn_latent", C.c_int32), ("gnn_iters", C.c_int32), ("edge_enc_input", C.c_int32),
                ("threshold", C.c_float), ("precision", C.c_int32), ("engine", C.c_int32),
                ("max_events", C.c_int32), ("max_hits", C.c_int32), ("validate_input", C.c_int32),
                ("emb_input", C.c_int32), ("cyl_offset", C.c_float * 3), ("cyl_div", C.c_float * 3),
                ("state_dtype", C.c_int32), ("max_triplets", C.c_int32), ("triplet_threshold", C.c_float),
                ("alloc", ALLOC_FN), ("dealloc", DEALLOC_FN), ("alloc_ctx", C.c_void_p)]


class EtxOutput(C.Structure):
    _fields_ = [("d_edge_src", C.c_void_p), ("d_edge_dst", C.c_void_p), ("d_edge_score", C.c_void_p),
                ("d_edge_logit", C.c_void_p), ("d_track_id", C.c_void_p), ("d_n_edges", C.c_void_p),
                ("h_n_edges", C.POINTER(C.c_int32)), ("n_hits", C.c_int32)]


class EtxTracks(C.Structure):
    _fields_ = [("d_track_index", C.c_void_p), ("d_track_offsets", C.c_void_p), ("d_track_hits", C.c_void_p),
                ("d_event_track_offsets", C.c_void_p), ("d_n_tracks", C.c_void_p), ("h_n_tracks", C.POINTER(C.c_int32))]


class EtxTriplets(C.Structure):
    _fields_ = [("d_first", C.c_void_p * 3), ("d_second", C.c_void_p * 3), ("d_hit", C.c_void_p * 3),
                ("d_logit", C.c_void_p * 3), ("d_score", C.c_void_p * 3), ("d_count", C.c_void_p),
                ("h_count", C.POINTER(C.c_int32)), ("capacity", C.c_int32)]


class EtxTripletComponents(C.Structure):
    _fields_ = [("d_edge_component", C.c_void_p), ("d_shared", C.c_void_p), ("d_n_shared", C.c_void_p),
                ("h_n_shared", C.POINTER(C.c_int32)), ("capacity", C.c_int32)]


class EtxTripletTracks(C.Structure):
    _fields_ = [("d_track_offsets", C.c_void_p), ("d_track_hits", C.c_void_p), ("d_counts", C.c_void_p),
                ("h_counts", C.POINTER(C.c_int32)), ("track_capacity", C.c_int32), ("hit_capacity", C.c_int32)]


class Inject(C.Structure):
    _fields_ = [("d_emb", C.c_void_p), ("d_src", C.c_void_p), ("d_dst", C.c_void_p), ("n_edges", C.c_int32),
                ("d_logit", C.c_void_p), ("last_stage", C.c_int32)]


def lib_path() -> str:
    return _LIB_PATH


def declared_symbols() -> list[str]:
    """Every function include/etx.h declares (used by the CPU test that checks the exports)."""
    text = open(_HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(etx_[a-z_0-9]+)\s*\(", text)))


_lib = None


def load_library():
    """dlopen libetx.so and declare the signatures.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2407_12119_b200._build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(_LIB_PATH)
    vp, i32p, f32p = C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_float)
    L.etx_create.restype = C.c_int
    L.etx_create.argtypes = [vp, C.c_size_t, C.POINTER(Hyperparams), C.POINTER(vp)]
    L.etx_run.restype = C.c_int
    L.etx_run.argtypes = [vp, vp, vp, i32p, C.c_int32, vp, C.POINTER(EtxOutput)]
    L.etx_run_host.restype = C.c_int
    L.etx_run_host.argtypes = [vp, vp, vp, i32p, C.c_int32, vp, vp, vp, vp, vp, i32p]
    L.etx_destroy.restype = C.c_int
    L.etx_destroy.argtypes = [vp]
    L.etx_submit_host.restype = C.c_int
    L.etx_submit_host.argtypes = [vp, vp, vp, i32p, C.c_int32, vp, vp, vp, vp, vp, vp, i32p]
    L.etx_wait_host.restype = C.c_int
    L.etx_wait_host.argtypes = [vp, C.c_int32]
    L.etx_triplets.restype = C.c_int
    L.etx_triplets.argtypes = [vp, vp, C.POINTER(EtxTriplets)]
    L.etx_triplet_components.restype = C.c_int
    L.etx_triplet_components.argtypes = [vp, vp, C.POINTER(EtxTripletComponents)]
    L.etx_triplet_tracks.restype = C.c_int
    L.etx_triplet_tracks.argtypes = [vp, C.c_int32, vp, C.POINTER(EtxTripletTracks)]
    L.etx_calibrate.restype = C.c_int
    L.etx_calibrate.argtypes = [vp, vp, vp, i32p, C.c_int32, vp, f32p, C.c_int32, i32p]
    L.etx_input_status.restype = C.c_int
    L.etx_input_status.argtypes = [vp]
    L.etx_tracks.restype = C.c_int
    L.etx_tracks.argtypes = [vp, C.c_int32, vp, C.POINTER(EtxTracks)]
    L.etx_tracks_static.restype = C.c_int
    L.etx_tracks_static.argtypes = [vp, vp, C.c_int32, C.c_int32, C.c_int32, vp, vp, vp, vp, vp, vp]
    L.etx_tracks_static_error.restype = C.c_char_p
    L.etx_tracks_static_error.argtypes = []
    L.etx_workspace_bytes.restype = C.c_size_t
    L.etx_workspace_bytes.argtypes = [vp]
    L.etx_status_string.restype = C.c_char_p
    L.etx_status_string.argtypes = [C.c_int]
    L.etx_last_error.restype = C.c_char_p
    L.etx_last_error.argtypes = [vp]
    L.etx_dbg_run.restype = C.c_int
    L.etx_dbg_run.argtypes = [vp, vp, vp, i32p, C.c_int32, vp, C.POINTER(Inject), C.POINTER(EtxOutput)]
    L.etx_dbg_buffer.restype = C.c_int
    L.etx_dbg_buffer.argtypes = [vp, C.c_char_p, C.POINTER(vp), C.POINTER(C.c_size_t)]
    L.etx_dbg_tap_layer.restype = C.c_int
    L.etx_dbg_tap_layer.argtypes = [vp, C.c_int32]
    L.etx_dbg_enable_timing.restype = C.c_int
    L.etx_dbg_enable_timing.argtypes = [vp, C.c_int32]
    L.etx_dbg_stage_times.restype = C.c_int
    L.etx_dbg_stage_times.argtypes = [vp, f32p]
    L.etx_dbg_launch_count.restype = C.c_int64
    L.etx_dbg_launch_count.argtypes = [vp]
    _lib = L
    return L


def lib():
    return load_library()


TRACKS_STATIC_MAX_HITS = 1 << 20        # ETX_TRACKS_STATIC_MAX_HITS of include/etx.h


def tracks_static(d_track_id, d_event_offsets, min_hits: int, out: dict) -> None:
    """etx_tracks_static on the current stream: the regrouping of `Etx.tracks` without a handle, for callers that may
    not allocate device memory (the library takes its work arrays from a fixed array inside libetx.so, see
    include/etx.h).  Every tensor is the caller's: `d_track_id` [n_hits] and `d_event_offsets` [n_events + 1] are int32
    CUDA tensors, `out` holds int32 CUDA tensors track_index [n_hits], track_offsets [n_hits + 1], track_hits [n_hits],
    event_track_offsets [n_events + 1] and n_tracks [1], which the call fills.  Nothing is allocated here either and
    nothing is synchronised.  Calls that could overlap on one GPU must be ordered by the caller."""
    import torch
    L = load_library()
    n_hits, n_events = int(d_track_id.numel()), int(d_event_offsets.numel()) - 1
    for name, t, n in (("track_id", d_track_id, n_hits), ("event_offsets", d_event_offsets, n_events + 1),
                       ("track_index", out["track_index"], n_hits), ("track_offsets", out["track_offsets"], n_hits + 1),
                       ("track_hits", out["track_hits"], n_hits), ("event_track_offsets", out["event_track_offsets"], n_events + 1),
                       ("n_tracks", out["n_tracks"], 1)):
        if not (t.is_cuda and t.dtype == torch.int32 and t.is_contiguous() and t.numel() >= n):
            raise ValueError(f"tracks_static: {name} must be a contiguous int32 CUDA tensor with at least {n} elements")
    st = L.etx_tracks_static(d_track_id.data_ptr(), d_event_offsets.data_ptr(), n_hits, n_events, int(min_hits),
                             C.c_void_p(torch.cuda.current_stream().cuda_stream), out["track_index"].data_ptr(),
                             out["track_offsets"].data_ptr(), out["track_hits"].data_ptr(),
                             out["event_track_offsets"].data_ptr(), out["n_tracks"].data_ptr())
    if st != 0:
        raise EtxError(st, L.etx_tracks_static_error().decode())


def hyperparams_from_config(cfg, max_events: int, max_hits: int, precision: str | None = None,
                            engine: str = "auto", validate_input: bool = False, n_planes: int = 26, max_triplets: int = 0, state_dtype: str | None = None,
                            norm_offset=(0.0, 0.0, 300.0), norm_div=(40.0, 40.0, 1050.0),
                            cyl_offset=(-20.0, 0.0, 300.0), cyl_div=(12.0, 3.14159274, 1050.0)) -> Hyperparams:
    """etx_hyperparams from a datagen.EtxConfig-like object (attribute access only)."""
    hp = Hyperparams()
    hp.struct_size = C.sizeof(Hyperparams)
    hp.n_planes = n_planes
    hp.norm_offset = (C.c_float * 3)(*norm_offset)
    hp.norm_div = (C.c_float * 3)(*norm_div)
    hp.emb_hidden, hp.emb_n_hidden_layers, hp.emb_dim = cfg.emb_hidden, cfg.emb_n_hidden_layers, cfg.emb_dim
    hp.k, hp.window = cfg.k, cfg.window
    hp.d2_max = cfg.d2_max if math.isfinite(cfg.d2_max) else float("inf")
    hp.gnn_latent, hp.gnn_iters, hp.edge_enc_input = cfg.gnn_latent, cfg.gnn_iters, cfg.edge_enc_input
    hp.threshold = cfg.threshold
    hp.precision = PRECISION[precision or cfg.precision]
    hp.engine = ENGINE[engine]
    hp.max_events, hp.max_hits = max_events, max_hits
    hp.validate_input = int(validate_input)
    hp.emb_input = getattr(cfg, "emb_input", 0)
    hp.cyl_offset = (C.c_float * 3)(*cyl_offset)
    hp.cyl_div = (C.c_float * 3)(*cyl_div)
    hp.state_dtype = STATE_DTYPE[state_dtype if state_dtype is not None else getattr(cfg, "state_dtype", "auto")]
    hp.max_triplets = int(max_triplets)
    hp.triplet_threshold = float(getattr(cfg, "triplet_threshold", 0.5))
    return hp


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2407_12119_b200 needs a CUDA device (no CPU fallback)")
    return torch


class Etx:
    """One etx_handle.  Methods mirror the C entry points; tensors are torch CUDA tensors used as plain
    device buffers, the stream is torch's current stream."""

    def __init__(self, blob: bytes, hp: Hyperparams):
        self._L = load_library()
        _torch()
        self._h = C.c_void_p()
        self.hp = hp
        self._blob = bytes(blob)
        st = self._L.etx_create(self._blob, len(self._blob), C.byref(hp), C.byref(self._h))
        if st != 0:
            self._h = C.c_void_p()
            raise EtxError(st, "etx_create")
        self._keep = None

    # -- lifetime -------------------------------------------------------------------------------
    def destroy(self):
        if getattr(self, "_h", None) and self._h.value:
            self._L.etx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _check(self, st: int, what: str):
        if st != 0:
            raise EtxError(st, f"{what}: {self._L.etx_last_error(self._h).decode()}")

    @staticmethod
    def _stream():
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)

    @staticmethod
    def _offsets(event_offsets):
        import numpy as np
        eo = np.ascontiguousarray(event_offsets, dtype=np.int32)
        return eo, eo.ctypes.data_as(C.POINTER(C.c_int32)), int(eo.size - 1)

    # -- the three-call contract ----------------------------------------------------------------
    def run(self, d_xyz, d_plane, event_offsets) -> EtxOutput:
        """etx_run: enqueue on the current stream; returns the raw output struct (device pointers)."""
        eo, eop, B = self._offsets(event_offsets)
        out = EtxOutput()
        self._keep = (d_xyz, d_plane, eo)
        st = self._L.etx_run(self._h, C.c_void_p(d_xyz.data_ptr()), C.c_void_p(d_plane.data_ptr()), eop, B,
                             self._stream(), C.byref(out))
        self._check(st, "etx_run")
        return out

    def input_status(self) -> int:
        """etx_input_status: verdict of the device-side input validation of the last completed run (0 = ETX_OK)."""
        return int(self._L.etx_input_status(self._h))

    def run_host(self, h_xyz, h_plane, event_offsets, h_score, h_src, h_dst, h_track_id) -> int:
        """etx_run_host: host (ideally pinned) tensors in and out; synchronises; returns E."""
        eo, eop, B = self._offsets(event_offsets)
        E = C.c_int32(0)
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p()
        st = self._L.etx_run_host(self._h, ptr(h_xyz), ptr(h_plane), eop, B, self._stream(), ptr(h_score),
                                  ptr(h_src), ptr(h_dst), ptr(h_track_id), C.byref(E))
        self._check(st, "etx_run_host")
        return int(E.value)

    def submit_host(self, h_xyz, h_plane, event_offsets, h_score, h_src, h_dst, h_track_id, h_n_edges) -> int:
        """etx_submit_host: pinned host tensors in and out, returns at once with a ticket (two may be in flight)."""
        eo, eop, B = self._offsets(event_offsets)
        t = C.c_int32(0)
        ptr = lambda x: C.c_void_p(x.data_ptr()) if x is not None else C.c_void_p()
        self._keep_async = getattr(self, "_keep_async", [])[-3:] + [(h_xyz, h_plane, eo, h_score, h_src, h_dst, h_track_id, h_n_edges)]
        st = self._L.etx_submit_host(self._h, ptr(h_xyz), ptr(h_plane), eop, B, self._stream(), ptr(h_score), ptr(h_src),
                                     ptr(h_dst), ptr(h_track_id), ptr(h_n_edges), C.byref(t))
        self._check(st, "etx_submit_host")
        return int(t.value)

    def wait_host(self, ticket: int):
        self._check(self._L.etx_wait_host(self._h, int(ticket)), "etx_wait_host")

    # -- debug entry points ----------------------------------------------------------------------
    def dbg_run(self, d_xyz, d_plane, event_offsets, emb=None, src=None, dst=None, logit=None,
                last_stage: int = 5) -> EtxOutput:
        eo, eop, B = self._offsets(event_offsets)
        inj = Inject()
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p()
        inj.d_emb, inj.d_src, inj.d_dst, inj.d_logit = ptr(emb), ptr(src), ptr(dst), ptr(logit)
        inj.n_edges = int(src.numel()) if src is not None else 0
        inj.last_stage = last_stage
        out = EtxOutput()
        self._keep = (d_xyz, d_plane, eo, emb, src, dst, logit)
        st = self._L.etx_dbg_run(self._h, ptr(d_xyz), ptr(d_plane), eop, B, self._stream(), C.byref(inj), C.byref(out))
        self._check(st, "etx_dbg_run")
        return out

    def tap_layer(self, index: int):
        self._check(self._L.etx_dbg_tap_layer(self._h, index), "etx_dbg_tap_layer")

    def enable_timing(self, on: bool = True):
        self._check(self._L.etx_dbg_enable_timing(self._h, int(on)), "etx_dbg_enable_timing")

    def stage_times(self) -> dict:
        arr = (C.c_float * len(STAGE_NAMES))()
        self._check(self._L.etx_dbg_stage_times(self._h, arr), "etx_dbg_stage_times")
        return {n: float(v) for n, v in zip(STAGE_NAMES, arr)}

    def tracks(self, n_hits: int, n_events: int, min_hits: int = 3) -> dict:
        """etx_tracks on the current stream after a run over (n_events, n_hits); synchronises, returns torch tensors."""
        import torch
        out = EtxTracks()
        self._check(self._L.etx_tracks(self._h, int(min_hits), self._stream(), C.byref(out)), "etx_tracks")
        torch.cuda.current_stream().synchronize()
        T = int(out.h_n_tracks[0])
        offs = self._copy_out(out.d_track_offsets, 4 * (T + 1), torch.int32)
        n_hits_kept = int(offs[-1].item()) if T else 0
        return dict(n_tracks=T, track_offsets=offs,
                    track_index=self._copy_out(out.d_track_index, 4 * n_hits, torch.int32),
                    track_hits=self._copy_out(out.d_track_hits, 4 * n_hits_kept, torch.int32),
                    event_track_offsets=self._copy_out(out.d_event_track_offsets, 4 * (n_events + 1), torch.int32))

    def triplets(self) -> dict:
        """etx_triplets on the current stream after a run; synchronises.  -> {kind: dict(first, second, hit, logit, score)}
        as torch tensors, plus "count" (the true counts) and "capacity"."""
        import torch
        out = EtxTriplets()
        self._check(self._L.etx_triplets(self._h, self._stream(), C.byref(out)), "etx_triplets")
        torch.cuda.current_stream().synchronize()
        res = {"count": [int(out.h_count[k]) for k in range(3)], "capacity": int(out.capacity)}
        for k, kind in enumerate(("articulation", "left_elbow", "right_elbow")):
            n = min(res["count"][k], res["capacity"])
            res[kind] = dict(first=self._copy_out(out.d_first[k], 4 * n, torch.int32), second=self._copy_out(out.d_second[k], 4 * n, torch.int32),
                             hit=self._copy_out(out.d_hit[k], 4 * n, torch.int32), logit=self._copy_out(out.d_logit[k], 4 * n, torch.float32),
                             score=self._copy_out(out.d_score[k], 4 * n, torch.float32))
        return res

    def triplet_components(self, n_edges: int) -> dict:
        """etx_triplet_components after triplets(); synchronises.  -> dict(edge_component [E], shared [n, 2])."""
        import torch
        out = EtxTripletComponents()
        self._check(self._L.etx_triplet_components(self._h, self._stream(), C.byref(out)), "etx_triplet_components")
        torch.cuda.current_stream().synchronize()
        n = min(int(out.h_n_shared[0]), int(out.capacity))
        return dict(edge_component=self._copy_out(out.d_edge_component, 4 * n_edges, torch.int32),
                    shared=self._copy_out(out.d_shared, 8 * n, torch.int32).reshape(-1, 2), n_shared=int(out.h_n_shared[0]))

    def triplet_tracks(self, min_hits: int = 3) -> dict:
        """etx_triplet_tracks after triplet_components(); synchronises.  -> dict(track_offsets [T + 1], track_hits,
        n_tracks, n_listed_hits, overflow); the lists are cut at the capacities when overflow is set."""
        import torch
        out = EtxTripletTracks()
        self._check(self._L.etx_triplet_tracks(self._h, int(min_hits), self._stream(), C.byref(out)), "etx_triplet_tracks")
        torch.cuda.current_stream().synchronize()
        T, H, ovf = int(out.h_counts[0]), int(out.h_counts[1]), int(out.h_counts[2])
        Tl, Hl = min(T, int(out.track_capacity)), min(H, int(out.hit_capacity))
        return dict(n_tracks=T, n_listed_hits=H, overflow=ovf,
                    track_offsets=self._copy_out(out.d_track_offsets, 4 * (Tl + 1), torch.int32),
                    track_hits=self._copy_out(out.d_track_hits, 4 * Hl, torch.int32))

    def calibrate(self, d_xyz, d_plane, event_offsets):
        """etx_calibrate on the current stream (an ETX_FP32 handle): the INT8 activation scales, one per quantised Linear
        in blob order, as a numpy float32 array -- what datagen.pack_blob(cfg, layers, scales) appends to the blob."""
        import numpy as np
        eo, eop, B = self._offsets(event_offsets)
        n = C.c_int32(0)
        self._check(self._L.etx_calibrate(self._h, None, None, eop, B, self._stream(), None, 0, C.byref(n)), "etx_calibrate")
        scales = np.zeros(int(n.value), np.float32)
        self._check(self._L.etx_calibrate(self._h, C.c_void_p(d_xyz.data_ptr()), C.c_void_p(d_plane.data_ptr()), eop, B, self._stream(),
                                          scales.ctypes.data_as(C.POINTER(C.c_float)), int(n.value), C.byref(n)), "etx_calibrate")
        return scales

    def workspace_bytes(self) -> int:
        return int(self._L.etx_workspace_bytes(self._h))

    def launch_count(self) -> int:
        return int(self._L.etx_dbg_launch_count(self._h))

    def buffer(self, name: str, dtype, shape=None):
        """A torch copy of an internal device buffer of the last run; synchronises."""
        import torch
        torch.cuda.current_stream().synchronize()
        p, n = C.c_void_p(), C.c_size_t()
        self._check(self._L.etx_dbg_buffer(self._h, name.encode(), C.byref(p), C.byref(n)), "etx_dbg_buffer")
        return self._copy_out(p.value, n.value, dtype, shape)

    def buffer_view(self, name: str, dtype):
        """A zero-copy, WRITABLE torch view of an internal device buffer (etx_dbg_buffer).  For fault-injection and
        fixture tests only: it aliases library-owned memory."""
        import torch
        torch.cuda.current_stream().synchronize()
        p, n = C.c_void_p(), C.c_size_t()
        self._check(self._L.etx_dbg_buffer(self._h, name.encode(), C.byref(p), C.byref(n)), "etx_dbg_buffer")

        class _Raw:
            __cuda_array_interface__ = {"shape": (int(n.value),), "typestr": "|u1", "data": (int(p.value), False), "version": 2}
        return torch.as_tensor(_Raw(), device="cuda").view(dtype)

    @staticmethod
    def _copy_out(ptr, nbytes: int, dtype, shape=None):
        """Clone `nbytes` of library-owned device memory into a fresh torch tensor of `dtype`."""
        import torch
        if not nbytes:
            out = torch.empty(0, dtype=dtype, device="cuda")
        else:
            class _Raw:     # zero-copy view of the raw pointer through the CUDA array interface
                __cuda_array_interface__ = {"shape": (int(nbytes),), "typestr": "|u1", "data": (int(ptr), False), "version": 2}
            out = torch.as_tensor(_Raw(), device="cuda").clone().view(dtype)
        return out.view(shape) if shape is not None else out

    def results(self, out: EtxOutput) -> dict:
        """Synchronise and copy the outputs of a run into torch tensors."""
        import torch
        torch.cuda.current_stream().synchronize()
        E, N = int(out.h_n_edges[0]), int(out.n_hits)
        return dict(n_edges=E,
                    src=self._copy_out(out.d_edge_src, 4 * E, torch.int32),
                    dst=self._copy_out(out.d_edge_dst, 4 * E, torch.int32),
                    score=self._copy_out(out.d_edge_score, 4 * E, torch.float32),
                    logit=self._copy_out(out.d_edge_logit, 4 * E, torch.float32),
                    track_id=self._copy_out(out.d_track_id, 4 * N, torch.int32))
