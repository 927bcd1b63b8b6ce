#!/usr/bin/env python
"""bench.py -- throughput of the ETX4VELO hot path (S0..S5) on synthetic VELO-shaped events.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg2] [--engine auto|simt] [--streams S]
    python bench.py --impl reference ...        # the CPU oracle on a bounded sample of the same workload

One "step" = one pass of the whole hot path over one batch (BASELINE.json configs[2]: 500 events at
pile-up 5, bf16 MLPs).  `value` is events/s with inputs resident in HBM; `e2e` is the same metric through
etx_run_host with pinned HOST buffers (H2D + D2H inside the timed region).  `roofline` describes the
dominant kernel (the edge network, S4e), timed live with CUDA events on the launching stream.  N > 1:
one process per GPU (torchrun), each rank runs its own batch, no collective on the data path (events are
independent) -- weak scaling.  DESIGN.md sec. 7 states every formula used here.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import datagen  # noqa: E402

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel (S4e edge network): the mean over the
# six launches of one pass (five write e back, the last does not), from the ncu pass over this very command summarised
# in profiles/r3_launches_cfg2.md (15,061.8 MB / 6; round 2's --set full capture gave 2.5139e9), per workload; bench.py
# cannot run ncu itself.
NCU_TRAFFIC_BYTES = {("cfg2", 500): 2.5103e9}
METRIC = "events_per_s"
UNIT = "events/s"
DTYPE = {"fp32": "f32", "bf16": "bf16", "int8": "int8"}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]), bf16_sustained=float(d["bf16_tflops_sustained"]),
                    source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler(threading.Thread):
    """SM clock + throttle reasons during the timed region (B200_PROFILING.md recipe): NVML in-process every 5 ms
    (pynvml), falling back to polling nvidia-smi, which manages only a sample or two in a 0.2 s region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4))

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self._stop_evt = index, [], threading.Event()
        self.sm, self.sm_max, self.reasons, self.nvml = [], None, set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].strip().isdigit() else index
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def run(self):
        while not self._stop_evt.is_set():
            try:
                if self.nvml is not None:
                    self.sm.append(float(self.nvml.nvmlDeviceGetClockInfo(self.handle, self.nvml.NVML_CLOCK_SM)))
                    try:
                        mask = int(self.nvml.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
                    except Exception:
                        mask = int(self.nvml.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
                    self.reasons.update(name for name, bit in self.REASONS if mask & bit)
                    self._stop_evt.wait(0.005)
                    continue
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    f = [x.strip() for x in out.split(",")]
                    if f[0].replace(".", "").isdigit():
                        self.sm.append(float(f[0]))
                    if f[1].replace(".", "").isdigit():
                        self.sm_max = max(self.sm_max or 0.0, float(f[1]))
                    self.reasons.update(name for (name, _), v in zip(self.REASONS, (f[3], f[4], f[5], f[6])) if v.lower().startswith("active"))
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons), "samples": len(self.sm), "source": "nvml" if self.nvml is not None else "nvidia-smi"}


def workload(cfg, rank: int, world: int = 1):
    from paper_2407_12119_b200.sharding import rank_events
    first, n = rank_events(rank, world, cfg.n_events)
    batch = datagen.generate_batch(cfg, n_events=n, first_event=first)
    layers = datagen.make_weights(cfg, "he")                      # BASELINE.json: He-uniform, zero bias
    return batch, layers


def calibration_batch():
    return datagen.generate_batch(datagen.get_config("cfg1"), n_events=datagen.configs.CALIBRATION_EVENTS,
                                  seed=datagen.configs.CALIBRATION_SEED)


def int8_scales(cfg, layers):
    """INT8 activation scales from the library's own calibration call (etx_calibrate: the fp32 FFMA engine over the
    16-event calibration batch); part of producing the blob, not of the timed path (R21)."""
    import torch
    import paper_2407_12119_b200 as etx
    cal = calibration_batch()
    cfg32 = cfg.replace(precision="fp32", state_dtype="auto")
    hp = etx.hyperparams_from_config(cfg32, cal.n_events, cal.n_hits)
    ctx = etx.Etx(datagen.pack_blob(cfg32, layers), hp)
    scales = ctx.calibrate(torch.from_numpy(cal.xyz).cuda(), torch.from_numpy(cal.plane).cuda(), cal.event_offsets)
    ctx.destroy()
    return scales


def int8_scales_reference(cfg, layers):
    """The reference arm has no GPU library: the oracle's own calibration (the same definition, R21)."""
    import oracle
    cal = calibration_batch()
    return oracle.calibrate_int8(datagen.pack_blob(cfg, layers), cal.xyz, cal.plane, cal.event_offsets, cfg.k, cfg.window)


def stage_model(cfg, N, E, pairs, peaks):
    """Algorithmic bytes / flops per step for every stage -> {stage: (bound, work, peak, unit)}."""
    D, H, d, L, k = cfg.emb_hidden, cfg.emb_n_hidden_layers, cfg.gnn_latent, cfg.gnn_iters, cfg.k
    b = 2 if (cfg.precision == "bf16" or (cfg.precision == "int8" and getattr(cfg, "state_dtype", "auto") == "bf16")) else 4
    tens = peaks["bf16_sustained"] * (2.0 if cfg.precision == "int8" else 1.0)      # int8 nominal = 2x bf16
    ffma = 148 * 128 * 2 * 1.965e9 / 1e12                                           # TFLOP/s at max clock
    mlp_peak, mlp_bound = (ffma, "alu") if cfg.precision == "fp32" else (tens, "tensor")
    alu_lane = 148 * 128 * 1.965e9                                                  # lane-instructions / s
    return {
        "S0_plane_offsets": ("hbm", 16.0 * N + 4.0 * N, peaks["hbm"], "GB/s"),
        "S1_embedding": (mlp_bound, N * 2.0 * (3 * D + (H - 1) * D * D + 4 * D), mlp_peak, "TFLOP/s"),
        "S2_knn": ("alu", pairs * 12.0, alu_lane, "lane-instr/s"),
        "S3_compaction_csc": ("hbm", 4.0 * k * N + 12.0 * E + 8.0 * E + 16.0 * N, peaks["hbm"], "GB/s"),
        # the stage only writes the state: bound by the (N + E) d b bytes of h0 / e0 (profiles/r1f), not by its FLOPs
        "S4_encoders": ("hbm", 1.0 * (N + E) * d * b + 16.0 * N + 8.0 * E, peaks["hbm"], "GB/s") if cfg.precision != "fp32"
                       else (mlp_bound, 2.0 * (3 * d + d * d) * (N + E), mlp_peak, "TFLOP/s"),
        # e is read from HBM once (the second direction finds its rows in L2: ncu, profiles/r1f_stage_rooflines.md)
        "S4c_scatter": ("hbm", L * (1.0 * E * d * b + 2.0 * N * d * b + 4.0 * E + 8.0 * N), peaks["hbm"], "GB/s"),
        # fp32 mode runs the networks on the FFMA pipe in the pinned order: bound by their FLOPs, not by bytes
        "S4d_node_net": ("hbm", L * (4.0 * N * d * b), peaks["hbm"], "GB/s") if cfg.precision != "fp32"
                        else ("alu", L * 2.0 * (3 * d * d + d * d) * N, ffma, "TFLOP/s"),
        # e is read by every step and written by all but the last (e^L feeds only the classifier, which is fused)
        "S4e_edge_net_head": ("hbm", L * ((2.0 * d * b + 8.0) * E + N * d * b) + 8.0 * E - (E * d * b if L else 0.0),
                              peaks["hbm"], "GB/s") if cfg.precision != "fp32"
                             else ("alu", (L * 2.0 * (3 * d * d + d * d) + 2.0 * d) * E, ffma, "TFLOP/s"),
        "S5_components": ("hbm", 12.0 * E + 8.0 * N, peaks["hbm"], "GB/s"),
    }


def run_oracle_sample(cfg, batch, layers, n_events, scales=None):
    import oracle
    sub = batch.slice_events(0, min(n_events, batch.n_events))
    o = oracle.Oracle(datagen.pack_blob(cfg, layers, scales), cfg.precision, state_dtype=getattr(cfg, "state_dtype", "auto"))
    t0 = time.perf_counter()
    o.run(sub.xyz, sub.plane, sub.event_offsets, cfg.k, cfg.window, cfg.d2_max, cfg.threshold)
    dt = time.perf_counter() - t0
    return sub.n_events / dt, dt, sub.n_events, oracle.threads()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="etx", choices=["etx", "reference"])
    ap.add_argument("--config", default="cfg2")
    ap.add_argument("--events", type=int, default=None, help="override the batch size (debugging only)")
    ap.add_argument("--engine", default="auto", choices=["auto", "simt", "tc_serial"])
    ap.add_argument("--cpu-events", type=int, default=500, help="oracle sample size for cpu_baseline (about 10 s of CPU work at cfg2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--streams", type=int, default=1, help="handles on that many CUDA streams, each running the whole batch per step "
                    "(PAPER.md L223: Allen keeps several streams of 500 events in flight)")
    ap.add_argument("--stage-passes", type=int, default=5, help="instrumented passes the per-stage times are averaged over")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    cfg = datagen.get_config(args.config)
    if args.events:
        cfg = cfg.replace(n_events=args.events)
    config = {"workload": f"{cfg.name}: {cfg.n_events} synthetic VELO events/GPU, pile-up {cfg.mu_pv:g}, "
                          f"emb 3->{'->'.join([str(cfg.emb_hidden)] * cfg.emb_n_hidden_layers)}->4, k={cfg.k}, w={cfg.window}, "
                          f"d={cfg.gnn_latent}, L={cfg.gnn_iters}, {cfg.precision}"
                          + (f", d2_max={cfg.d2_max:g}" if cfg.d2_max != float("inf") else "")
                          + (", edge encoder on [h0_src,h0_dst]" if cfg.edge_enc_input else "")
                          + (", cylindrical embedding input" if cfg.emb_input else ""),
              "events_per_gpu": cfg.n_events, "weights": "He-uniform seed 7, zero bias"}

    # ------------------------------------------------------------------ reference arm = the CPU oracle
    if args.impl == "reference":
        if rank != 0:
            return 0
        batch, layers = workload(cfg, 0)
        scales = int8_scales_reference(cfg, layers) if cfg.precision == "int8" else None
        n_ev = max(1, min(args.cpu_events // 4, batch.n_events))
        for _ in range(min(args.warmup, 1)):
            run_oracle_sample(cfg, batch, layers, 1, scales)
        t_tot, ev_tot, cores = 0.0, 0, 1
        for _ in range(args.steps):
            _, dt, n, cores = run_oracle_sample(cfg, batch, layers, n_ev, scales)
            t_tot += dt; ev_tot += n
        value = ev_tot / t_tot
        hits = float(batch.event_offsets[n_ev]) / n_ev
        line = {"metric": METRIC, "value": value, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": DTYPE[cfg.precision], "data": "synthetic", "config": config,
                "hits_per_s": value * hits,
                "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                                 "sample": f"each step = the first {n_ev} events of the {cfg.n_events}-event batch, whole path S0..S5"},
                "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    # ------------------------------------------------------------------ the CUDA path
    import torch
    import paper_2407_12119_b200 as etx
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    batch, layers = workload(cfg, rank, world)
    scales = int8_scales(cfg, layers) if cfg.precision == "int8" else None
    blob = datagen.pack_blob(cfg, layers, scales)
    hp = etx.hyperparams_from_config(cfg, batch.n_events, batch.n_hits, engine=args.engine)
    ctx = etx.Etx(blob, hp)
    d_xyz = torch.from_numpy(batch.xyz).cuda()
    d_plane = torch.from_numpy(batch.plane).cuda()
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # further handles on their own streams (--streams): each runs the whole batch every step, concurrently
    extra = [(etx.Etx(blob, hp), torch.cuda.Stream()) for _ in range(max(args.streams, 1) - 1)]

    def one_step():
        o = ctx.run(d_xyz, d_plane, batch.event_offsets)
        for c2, s2 in extra:
            with torch.cuda.stream(s2):
                c2.run(d_xyz, d_plane, batch.event_offsets)
        return o

    def fork():                                    # the side streams start after everything already on the main stream
        for _, s2 in extra:
            s2.wait_stream(stream)

    def join():                                    # ... and the main stream ends after all of them
        for _, s2 in extra:
            stream.wait_stream(s2)

    fork()
    for _ in range(max(args.warmup, 3)):
        out = one_step()
    join()
    torch.cuda.synchronize()
    E = int(out.h_n_edges[0]); N = batch.n_hits
    d_, L_ = cfg.gnn_latent, cfg.gnn_iters
    sb = 2 if (cfg.precision == "bf16" or (cfg.precision == "int8" and getattr(cfg, "state_dtype", "auto") == "bf16")) else 4
    working_set = (E * d_ + 3 * N * d_) * sb + 12 * E + 32 * N           # e, h, m, edge list + scores, hit arrays
    L2_BYTES = 126e6
    flush_l2 = working_set < 2 * L2_BYTES
    if flush_l2:
        # the batch would stay (partly) resident in the 126 MB L2 from one step to the next: every step is timed on its
        # own and a 512 MB write in between evicts it (the write itself is outside the timed spans)
        flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
        config["l2"] = (f"per-step working set {working_set / 1e6:.0f} MB would fit the 126 MB L2: flushed between timed steps "
                        "(512 MB write, untimed; steps timed one by one)")
    else:
        config["l2"] = (f"per-step working set {working_set / 1e6:.0f} MB (edge state alone {E * d_ * sb / 1e6:.0f} MB) exceeds the "
                        "126 MB L2; no explicit flush")
    config["streams"] = max(args.streams, 1)
    sampler = ClockSampler(local_rank); sampler.start()
    launches0 = ctx.launch_count() + sum(c2.launch_count() for c2, _ in extra)
    barrier()
    if flush_l2:
        pairs_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for a, b_ in pairs_ev:
            flush_buf.fill_(1)
            a.record(stream); fork()
            out = one_step()
            join(); b_.record(stream)
        barrier()
        ms = sum(a.elapsed_time(b_) for a, b_ in pairs_ev)
    else:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream); fork()
        for _ in range(args.steps):
            out = one_step()
        join(); ev1.record(stream)
        barrier()
        ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop()
    launches = ctx.launch_count() + sum(c2.launch_count() for c2, _ in extra) - launches0
    for c2, _ in extra:
        c2.destroy()
    # per-stage times: extra passes of ONE handle with the library's stage events switched on (CUDA events on the
    # launching stream between the stages), averaged; the headline above is the plain etx_run path without them
    ctx.enable_timing(True)
    acc = {}
    n_pass = max(args.stage_passes, 1)
    for _ in range(n_pass):
        if flush_l2:
            flush_buf.fill_(1)
        ctx.run(d_xyz, d_plane, batch.event_offsets)
        torch.cuda.synchronize()
        for name, v in ctx.stage_times().items():
            acc.setdefault(name, []).append(v)
    stage_ms = {name: float(np.mean(v)) for name, v in acc.items()}
    stage_ms_spread = {name: [float(np.min(v)), float(np.max(v))] for name, v in acc.items()}
    ctx.enable_timing(False)
    from paper_2407_12119_b200.sharding import whole_job
    n_str = max(args.streams, 1)
    ms, (tot_events, tot_hits, _) = whole_job(ms, [batch.n_events * n_str, N * n_str, E], dist, "cuda")
    value = tot_events * args.steps / (ms * 1e-3)

    # ---- end to end through etx_run_host: pinned host buffers, H2D + D2H inside the timed region
    cap = cfg.k * N
    h_xyz = torch.from_numpy(batch.xyz).pin_memory(); h_plane = torch.from_numpy(batch.plane).pin_memory()
    h_score = torch.empty(max(cap, 1), dtype=torch.float32).pin_memory()
    h_src = torch.empty(max(cap, 1), dtype=torch.int32).pin_memory(); h_dst = torch.empty(max(cap, 1), dtype=torch.int32).pin_memory()
    h_tid = torch.empty(max(N, 1), dtype=torch.int32).pin_memory()
    ctx.run_host(h_xyz, h_plane, batch.event_offsets, h_score, h_src, h_dst, h_tid)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        E2 = ctx.run_host(h_xyz, h_plane, batch.event_offsets, h_score, h_src, h_dst, h_tid)
    torch.cuda.synchronize()
    e2e_sync_s = time.perf_counter() - t0
    e2e_sync_s, _ = whole_job(e2e_sync_s, [], dist, "cuda")
    # the same work through etx_submit_host / etx_wait_host: two batches in flight, so the H2D of step i + 1 and the
    # D2H of step i run under compute -- every step still copies its own inputs in and its own results out
    outs = [(h_score, h_src, h_dst, h_tid, torch.zeros(1, dtype=torch.int32)),
            (torch.empty_like(h_score).pin_memory(), torch.empty_like(h_src).pin_memory(), torch.empty_like(h_dst).pin_memory(),
             torch.empty_like(h_tid).pin_memory(), torch.zeros(1, dtype=torch.int32))]
    def pipelined(n):
        prev = None
        for i in range(n):
            o = outs[i & 1]
            t = ctx.submit_host(h_xyz, h_plane, batch.event_offsets, o[0], o[1], o[2], o[3], o[4])
            if prev is not None:
                ctx.wait_host(prev)
            prev = t
        ctx.wait_host(prev)
    pipelined(2)
    barrier()
    t0 = time.perf_counter()
    pipelined(args.steps)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s, _ = whole_job(e2e_s, [], dist, "cuda")
    assert int(outs[(args.steps - 1) & 1][4][0]) == E2
    e2e_events = tot_events / n_str                       # the end-to-end legs run one handle
    e2e = {"value": e2e_events * args.steps / e2e_s, "unit": UNIT,
           "h2d_bytes_per_step": int(16 * N + 4 * (batch.n_events + 1)), "d2h_bytes_per_step": int(12 * E2 + 4 * N + 4),
           "api": "etx_submit_host / etx_wait_host, two batches in flight (pinned host buffers; each step copies its inputs in and its results out)",
           "synchronous": {"value": e2e_events * args.steps / e2e_sync_s, "unit": UNIT, "api": "etx_run_host, one batch at a time"}}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- per-stage roofline fractions + the dominant kernel
    peaks = measured_peaks()
    po = batch.plane.astype(np.int64)
    pairs = 0
    for e in range(batch.n_events):
        cnt = np.bincount(po[batch.event_offsets[e]:batch.event_offsets[e + 1]], minlength=27)
        for w in range(1, cfg.window + 1):
            pairs += int((cnt[:26 - w] * cnt[w:26]).sum())
    model = stage_model(cfg, N, E, pairs, peaks)
    stages = {}
    for name, (bound, work, peak, unit) in model.items():
        t = stage_ms.get(name, 0.0) * 1e-3
        ach = (work / t / (1e12 if unit == "TFLOP/s" else 1e9 if unit == "GB/s" else 1.0)) if t > 0 else None
        stages[name] = {"ms": stage_ms.get(name, 0.0), "ms_min_max": stage_ms_spread.get(name), "bound": bound, "achieved": ach,
                        "peak": peak, "unit": unit, "frac": (ach / peak) if ach else None}
    dom = "S4e_edge_net_head"
    L = max(cfg.gnn_iters, 1)
    dom_ms = stage_ms[dom] / L
    dom_bound, _, dom_peak, dom_unit = model[dom]
    dom_div = 1e12 if dom_unit == "TFLOP/s" else 1e9
    wide = model[dom][1] / L                                  # every compulsory byte (or, fp32: the flops) per launch
    if dom_bound == "hbm":
        # e read + e write = 2 d b per edge, the h gathers L2-resident; the last launch of a pass
        # feeds only the fused classifier and does not write e back.  `frac` is quoted on THIS count; the wider one
        # (+ src / dst, h once per node, logit / score) is reported beside it.
        dom_bytes = (2 * L - 1) * d_ * sb * E / L
    else:
        dom_bytes = wide
    rate = lambda work: work / (dom_ms * 1e-3) / dom_div if dom_ms > 0 else None
    hbm_note = ("S4e moves its bytes once (ncu traffic / compulsory bytes = 0.98 at cfg2, 1.07 on the 8(d) count); what holds it below the copy peak is on chip: "
                "shared-memory bandwidth and the cp.async gather of h[src], h[dst] (profiles/r2_s4e_ablation.md)")
    roofline = {"kernel": "edge network MLP (S4e), one launch per message-passing step", "bound": dom_bound,
                "achieved": rate(dom_bytes), "peak": dom_peak, "unit": dom_unit,
                "frac": rate(dom_bytes) / dom_peak if dom_ms > 0 else None,
                "algorithmic_work_per_launch": dom_bytes,
                "algorithmic_count": "SURVEY.md sec. 8(d): 2 d b per edge (e read + e write), last launch of a pass writes no e"
                                     if dom_bound == "hbm" else "2 (3 d d + d d) flops per edge (+ 2 d for the head)",
                "compulsory": {"work_per_launch": wide, "achieved": rate(wide), "frac": rate(wide) / dom_peak if dom_ms > 0 else None,
                               "count": "algorithmic + src / dst (8 E) + h once per node (N d b) + logit and score writes"}
                              if dom_bound == "hbm" else None,
                "traffic": NCU_TRAFFIC_BYTES.get((cfg.name, cfg.n_events)) if n_str == 1 and args.engine == "auto" else None,
                "traffic_source": ("recorded: ncu dram__bytes_read.sum + dram__bytes_write.sum of this kernel at this workload (profiles/r3_launches_cfg2.md); "
                                   "bench.py cannot run ncu") if (cfg.name, cfg.n_events) in NCU_TRAFFIC_BYTES
                                  else "no ncu capture recorded for this workload",
                "note": hbm_note if dom_bound == "hbm" else "fp32 mode runs the networks on the FFMA pipe in the oracle's pinned order (DESIGN.md R4)",
                "l2": "flushed between steps" if flush_l2 else "working set exceeds L2",
                "peak_source": peaks["source"] if dom_bound == "hbm" else "derived: 148 SM x 128 lanes x 2 x 1.965 GHz (DESIGN.md sec. 3)",
                "avg_launch_ms": dom_ms, "stage_passes": n_pass,
                "share_of_step": stage_ms[dom] / (ms / args.steps / 1.0) if (ms > 0 and n_str == 1) else None}
    cpu_baseline = None
    if not args.no_cpu_baseline:
        v, dt, n, cores = run_oracle_sample(cfg, batch, layers, args.cpu_events, scales)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"first {n} events of the same batch, whole path S0..S5, {dt:.1f} s"}
        import oracle
        oracle.set_threads(1)                             # also once single-threaded, on a smaller sample
        v1, dt1, n1, _ = run_oracle_sample(cfg, batch, layers, max(1, args.cpu_events // 32), scales)
        oracle.set_threads(cores)
        cpu_baseline["single_thread"] = {"value": v1, "unit": UNIT, "cores": 1, "sample": f"first {n1} events, {dt1:.1f} s"}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": DTYPE[cfg.precision], "data": "synthetic", "config": config, "engine": args.engine,
            "hits_per_s": tot_hits * args.steps / (ms * 1e-3), "n_hits": N, "n_edges": E, "clocks": clocks, "e2e": e2e,
            "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu_baseline, "stages": stages}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
