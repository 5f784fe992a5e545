#!/usr/bin/env python
"""bench.py -- DDHF hot path on B200: NDFT Gterms/s and ms per 1280x720 window.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4|cfg5|cfg3|paper] [--impl reference]
                  [--no-sub] [--no-cpu-baseline] [--score-all] [--spectra]

A *step* is one pass of the whole hot path (a0-a8: ingest, NDFT power, spectral flatness, comb
score, mask, CCL/boxes) over one synthetic window.  Default workload: BASELINE.json config 4
(1280x720, 100 ms, ~10 M events, 5 % of the pixels hold 60 % of the events) -- the heaviest
single 1280x720 window; `--workload cfg5` runs the streaming config (sliding 50 ms windows,
10 ms hop, 50 Mev/s) with one step per window.

The default run (config 4, one GPU) also measures, each with its own clocks record, the variants
SURVEY.md section 8(d) lists: config 4 with the comb score on every active pixel, with Table 2's
thresholds, with the compact spectra written to HBM, config 5 (100 sliding windows, p50 / p99) and
the paper's own operating point -- the `sub` object of the line (`--no-sub` skips them).

Prints ONE JSON line (rank 0).  `value` = (pixel x frequency x event) terms of the active
pixels per step / device time per step, inputs resident in HBM.  `e2e` = the same through
ddhf_window_host(): pinned host events in, mask / boxes / counters back to the host, copies
inside the timed region.  `roofline` is for the fused NDFT+scoring kernel (FP32 ALU bound,
2 FMA = 4 flop per term); `cpu_baseline` is the float64 oracle timed on this box's host cores
on a bounded crop of the same window.

N > 1 (torchrun): every rank runs its own replica of the window (the path has no exchange
step: pixels and windows are independent), scaling = weak, value = sum over ranks / max time.
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

NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # 74.45: SMs x FP32 lanes x 2 flop x max SM clock
FLOP_PER_TERM = 4.0                                        # one complex phasor accumulate = 2 FMA
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_traffic.csv")   # dram__bytes per launch from committed ncu captures


def traffic_of(kernel_prefixes, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernels whose names start with
    one of `kernel_prefixes`, from the committed ncu summary of this build (profiles/r2_traffic.csv,
    written from `ncu --set full` / `--metrics dram__bytes_*` captures; profiles/r2_traffic.md names the
    commands).  None when the table has no row for the workload: nothing is guessed."""
    try:
        tot, hit = 0.0, False
        for line in open(TRAFFIC_CSV):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 4 and f[0] == workload and any(f[1].startswith(k) for k in kernel_prefixes):
                tot += float(f[2]) + float(f[3])
                hit = True
        return tot if hit else None
    except OSError:
        return None


class ClockSampler(threading.Thread):
    """Samples SM clock, power and throttle reasons through NVML while the timed region runs
    (every 2 ms; `nvidia-smi` takes ~100 ms per query, longer than a whole timed pass)."""

    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown"}

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index = index
        self.mhz: list[float] = []
        self.power: list[float] = []
        self.reasons: set[str] = set()
        self.max_mhz = None
        self.stop_flag = threading.Event()
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def sample(self):
        n = self.nvml
        self.mhz.append(float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM)))
        self.power.append(n.nvmlDeviceGetPowerUsage(self.handle) / 1000.0)
        bits = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
        for bit, name in self.REASONS.items():
            if bits & bit:
                self.reasons.add(name)

    def run(self):
        if self.nvml is None:
            return
        while not self.stop_flag.is_set():
            try:
                self.sample()
            except Exception:
                pass
            self.stop_flag.wait(0.002)

    def summary(self) -> dict:
        return {"sm_mhz": float(np.median(self.mhz)) if self.mhz else None, "sm_max_mhz": self.max_mhz,
                "power_w_max": float(max(self.power)) if self.power else None,
                "samples": len(self.mhz), "reasons": sorted(self.reasons),
                "source": "nvml" if self.nvml is not None else "unavailable"}


def load_workload(name: str):
    from paper_2603_08386_b200 import workloads
    if name == "cfg4":
        return workloads.make(4)
    if name == "cfg5":
        return workloads.make(5, n_windows=100)
    if name == "cfg3":
        return workloads.make(3)
    if name == "paper":                       # the paper's operating point on the config-4 scene
        return workloads.paper_native()
    raise SystemExit(f"unknown workload {name}")


def window_list(w, steps_needed: int):
    """(first event, count, t0) for each step."""
    if w.n_windows == 1:
        return [(0, len(w.events), w.t0_us)] * steps_needed
    wins = [w.window_slice(k) for k in range(w.n_windows)]
    return [wins[i % len(wins)] for i in range(steps_needed)]


def terms_of(res, n_freq: int, n_min: int) -> int:
    cnt = np.diff(res["row_ptr"])
    return int(cnt[cnt >= max(n_min, 1)].sum()) * n_freq


def oracle_sample(w, crop=(640, 360)):
    """Bounded sample of the workload for the CPU oracle: the top-left crop of the sensor."""
    cw, ch = min(crop[0], w.width), min(crop[1], w.height)
    lo, n, t0 = w.window_slice(0) if w.n_windows > 1 else (0, len(w.events), w.t0_us)
    ev = w.events[lo:lo + n]
    ev = ev[(ev["x"] < cw) & (ev["y"] < ch)]
    prm = dict(w.params, width=cw, height=ch)
    return prm, ev, t0, f"{cw}x{ch} crop (top-left) of the {w.width}x{w.height} window, {len(ev)} events"


def time_oracle(w, steps: int, warmup: int, crop=(320, 180)):
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import ddhf_oracle
    prm, ev, t0, what = oracle_sample(w, crop)
    times, terms = [], 0
    for i in range(warmup + steps):
        t = time.perf_counter()
        out = ddhf_oracle.window(prm, ev, t0, w.window_us, want_power=False)
        dt = time.perf_counter() - t
        if i >= warmup:
            times.append(dt)
        terms = terms_of(out, prm["n_freq"], prm["n_min"])
    return dict(value=terms / np.mean(times) / 1e9, unit="Gterms/s", cores=ddhf_oracle.num_threads(),
                kind="oracle", sample=what, ms_per_step=float(np.mean(times) * 1e3), terms_per_step=terms)


def aggregate_over_ranks(time_ms: float, units: float, world: int, device="cpu"):
    """Whole-job numbers of a replicas-only run: the slowest rank's time and the units of all ranks.
    The only data exchanged between ranks in this repository."""
    if world <= 1:
        return float(time_ms), float(units)
    import torch
    import torch.distributed as dist
    t = torch.tensor([time_ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([units], device=device, dtype=torch.float64)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def measure(w, *, steps, warmup, dev, world=1, local_rank=0, score_all=False, spectra=False, params=None, name="",
            slide=False, nufft=None):
    """Device-resident timing of `steps` windows of workload `w` (after `warmup`): whole-window CUDA-event
    time, per-stage times, clocks sampled during the timed region.  Returns (record, detector state)."""
    import torch
    import torch.distributed as dist
    from paper_2603_08386_b200 import binding
    prm = dict(params or w.params)
    # the stream stays resident; max_events = the largest window handed to ddhf_window
    max_ev = len(w.events) if w.n_windows == 1 else max(w.window_slice(k)[1] for k in range(w.n_windows))
    det = binding.Detector(prm, max_events=max_ev, score_all=score_all, timing=True, want_power=spectra, want_labels=False,
                           nufft=nufft is not None, nufft_min=int(nufft or 0), device=f"cuda:{local_rank}",
                           max_active=(prm["width"] * prm["height"]) if spectra else 1)
    d_ev = det.upload(w.events)
    wins = window_list(w, warmup + steps)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # one untimed pass to count the terms of every distinct window (device counters only tell
    # events and pixels; the term count needs the row lengths)
    terms_by_win = {}
    for lo, n, t0 in dict.fromkeys(wins):
        det.window(d_ev, n, t0, w.window_us, offset_events=lo)
        res = det.results()
        terms_by_win[(lo, n, t0)] = (terms_of(res, prm["n_freq"], prm["n_min"]), res)
    launches_per_window = binding.ddhf_launches_per_window(det.h)

    prev = {"hi": None, "t0": None}

    def run_window(lo, n, t0):
        """One step: ddhf_window on the slice, or (slide) ddhf_window_slide on the events that follow the
        previous step's slice; a step whose t0 does not continue the sequence restarts it from scratch."""
        if not slide:
            det.window(d_ev, n, t0, w.window_us, offset_events=lo)
            return
        hi = lo + n
        if prev["hi"] is not None and 0 <= t0 - prev["t0"] < w.window_us:
            det.slide(d_ev, hi - prev["hi"], t0, w.window_us, offset_events=prev["hi"])
        else:
            det.slide(d_ev, n, t0, w.window_us, offset_events=lo)
        prev["hi"], prev["t0"] = hi, t0

    for lo, n, t0 in wins[:warmup]:
        run_window(lo, n, t0)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    per_step_ms, stage = [], []
    # L2 hygiene: a step touches the events (16 B), the bucket-sorted items (4 B, written and read), csr_ev
    # (4 B) and the per-pixel maps.  When that is below twice the 126 MB L2, a 256 MB buffer is written
    # between steps (outside the timed intervals: one CUDA-event pair per step, their sum is the time).
    n_ev_step = max(n for _, n, _ in wins[warmup:])
    footprint = 28.0 * n_ev_step + 40.0 * prm["width"] * prm["height"]
    flush = footprint < 2 * 126e6
    scratch = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if flush else None
    if flush:
        pairs_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in wins[warmup:]]
        for (e0, e1), (lo, n, t0) in zip(pairs_ev, wins[warmup:]):
            scratch.fill_(1)
            e0.record()
            run_window(lo, n, t0)
            e1.record()
        barrier()
        total_ms = float(sum(e0.elapsed_time(e1) for e0, e1 in pairs_ev))
    else:
        ev0 = torch.cuda.Event(enable_timing=True)
        ev1 = torch.cuda.Event(enable_timing=True)
        ev0.record()
        for lo, n, t0 in wins[warmup:]:
            run_window(lo, n, t0)
        ev1.record()
        barrier()
        total_ms = ev0.elapsed_time(ev1)
    # per-step latency and per-stage split: a second timed pass with a sync per window
    for lo, n, t0 in wins[warmup:]:
        if flush:
            scratch.fill_(1)
        run_window(lo, n, t0)
        ms = det.stage_ms()
        stage.append(ms)
        per_step_ms.append(ms[4])
    sampler.stop_flag.set()
    sampler.join()
    stage = np.array(stage)
    terms_total = sum(terms_by_win[k][0] for k in wins[warmup:])
    total_ms, terms_all = aggregate_over_ranks(total_ms, terms_total, world, dev)
    res0 = terms_by_win[wins[warmup]][1]
    ndft_ms = float(stage[:, 1].mean())
    terms_per_step = terms_total / len(wins[warmup:])
    rec = {
        "name": name, "value": terms_all / (total_ms * 1e-3) / 1e9, "unit": "Gterms/s", "steps": steps, "warmup": warmup,
        "ms_per_step": total_ms / steps,
        "config": {"workload": f"{name}: {prm['width']}x{prm['height']} sensor, "
                               f"{w.window_us / 1e3:.1f} ms window, {res0['n_in']} events, "
                               f"{prm['n_freq']} bins, {prm['n_f0']} f0 candidates, H={prm['n_harm']}, "
                               f"n_min={prm['n_min']}, tau_sf={prm['tau_sf']}, tau_comb={prm['tau_comb']}",
                   "events_per_step": res0["n_in"], "active_pixels": res0["n_active"],
                   "scored_pixels": res0["n_scored"], "terms_per_step": terms_per_step,
                   "mask_pixels": int(res0["mask"].sum()), "boxes": res0["n_boxes"],
                   "score_all": bool(score_all), "spectra_to_hbm": bool(spectra),
                   "nufft_min_events": (None if nufft is None else (int(nufft) or 64)),
                   "ingest_mode": ("ddhf_window_slide: only the events that follow the previous window are sorted; the "
                                   "sequence restarts from scratch when the window list wraps around") if slide
                                  else "ddhf_window: every window bucketed from scratch",
                   "scoring_note": "the comb score is evaluated where SF <= tau_sf (PAPER.md L139 order) unless score_all: "
                                   "thresholds change the work done, not only the mask",
                   "l2": ("L2 flushed between steps (256 MB write, outside the timed intervals); step footprint %.0f MB"
                          if flush else "step footprint %.0f MB (events + bucket-sorted items + csr + maps) exceeds the 126 MB L2")
                         % (footprint / 1e6),
                   "replicas": world},
        "latency_ms": {"p50": float(np.percentile(per_step_ms, 50)), "p99": float(np.percentile(per_step_ms, 99)),
                       "ingest": float(stage[:, 0].mean()), "ndft": ndft_ms, "comb_score": float(stage[:, 2].mean()),
                       "ccl": float(stage[:, 3].mean())},
        # (with the NUFFT path the long rows do not execute their terms: no roofline fraction, and `value` is nominal)
        "ndft_frac_of_fp32_peak": None if nufft is not None else
                                  terms_per_step * FLOP_PER_TERM / (ndft_ms * 1e-3) / 1e12 / NOMINAL_FP32_TFLOPS,
        "clocks": sampler.summary(), "gpu_launches": launches_per_window * steps,
    }
    state = dict(det=det, d_ev=d_ev, wins=wins, terms_by_win=terms_by_win, stage=stage, terms_total=terms_total,
                 barrier=barrier, prm=prm, launches_per_window=launches_per_window)
    return rec, state


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sub", action="store_true", help="skip the variant measurements (the `sub` object)")
    ap.add_argument("--score-all", action="store_true", help="comb score on every active pixel (R14)")
    ap.add_argument("--spectra", action="store_true", help="also write the compact power spectra to HBM")
    ap.add_argument("--nufft", type=int, default=None, metavar="MIN",
                    help="rows of >= MIN events (0: the library default, 64) by the NUFFT path (DDHF_FLAG_NUFFT): approximate, "
                         "so the Gterms/s of such a run is nominal (terms of the direct sum it replaces / time)")
    ap.add_argument("--slide", action="store_true", help="streaming workloads: ddhf_window_slide (incremental CSR)")
    args = ap.parse_args()
    steps, warmup = max(args.steps, 1), max(args.warmup, 3 if args.impl == "ours" else 0)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        # The oracle, as it stands, on this box's host cores.  Rank 0 only.
        if rank != 0:
            return
        w = load_workload(args.workload)
        # every step is the oracle on a bounded sample (a crop of the window), so K steps stay within minutes
        r = time_oracle(w, steps, warmup)
        line = {"impl": "reference", "metric": "ndft_gterms_per_s", "value": r["value"], "unit": "Gterms/s",
                "n_gpus": args.gpus, "steps": steps, "warmup": warmup,
                "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"{args.workload} ({r['sample']})", "terms_per_step": r["terms_per_step"]},
                "cpu_baseline": {"value": r["value"], "unit": "Gterms/s", "cores": r["cores"],
                                 "kind": "oracle", "sample": r["sample"]},
                "e2e": {"value": r["value"], "unit": "Gterms/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return

    import torch
    import torch.distributed as dist
    from paper_2603_08386_b200 import binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the DDHF path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = load_workload(args.workload)
    rec, st = measure(w, steps=steps, warmup=warmup, dev=dev, world=world, local_rank=local_rank,
                      score_all=args.score_all, spectra=args.spectra, name=args.workload, slide=args.slide, nufft=args.nufft)
    det, wins, terms_by_win, stage, prm = st["det"], st["wins"], st["terms_by_win"], st["stage"], st["prm"]
    barrier = st["barrier"]

    # ---- end to end through the host-buffer entry points -------------------------------------------
    # e2e: ddhf_host_submit / ddhf_host_wait (two windows in flight: the 16 B/event host->device copy
    # of window i+1 overlaps the kernels of window i); every step copies its events from pinned host
    # memory and reads mask, boxes and counters back.  e2e_serial: ddhf_window_host, one window at a
    # time (copy, kernels, copy back, synchronise).
    NP = prm["width"] * prm["height"]
    h_ev = torch.from_numpy(np.ascontiguousarray(w.events).view(np.uint8).copy()).pin_memory()
    houts, hbufs = [], []
    for _ in range(2):
        t = (torch.zeros(NP, dtype=torch.uint8).pin_memory(),
             torch.zeros(det.cfg.max_boxes * 6, dtype=torch.int32).pin_memory(),
             torch.zeros(16, dtype=torch.int32).pin_memory())
        o = binding.DdhfHostOutputs()
        o.mask, o.boxes, o.counters = t[0].data_ptr(), t[1].data_ptr(), t[2].data_ptr()
        hbufs.append(t)
        houts.append(o)
    cst = torch.cuda.current_stream(dev).cuda_stream
    e2e_steps = steps
    e2e_wins = wins[warmup:warmup + e2e_steps]

    def run_pipelined(ws):
        for i, (lo, n, t0) in enumerate(ws):
            binding.ddhf_host_submit(det.h, h_ev.data_ptr() + 16 * lo, n, t0, w.window_us, houts[i & 1], cst)
            if i >= 1:
                binding.ddhf_host_wait(det.h)
        binding.ddhf_host_wait(det.h)

    def run_serial(ws):
        for lo, n, t0 in ws:
            binding.ddhf_window_host(det.h, h_ev.data_ptr() + 16 * lo, n, t0, w.window_us, houts[0], cst)

    # the same stream as 8-byte events (ddhf_event8: nothing is lost, results are bit-identical)
    from paper_2603_08386_b200 import workloads as _wl
    t_base = int(w.events["t"].min()) if len(w.events) else 0
    h_ev8 = torch.from_numpy(_wl.pack_events(w.events, t_base).view(np.uint8).copy()).pin_memory()

    def run_packed(ws):
        for i, (lo, n, t0) in enumerate(ws):
            binding.ddhf_host_submit_packed(det.h, h_ev8.data_ptr() + 8 * lo, n, t_base, t0, w.window_us, houts[i & 1], cst)
            if i >= 1:
                binding.ddhf_host_wait(det.h)
        binding.ddhf_host_wait(det.h)

    e2e_terms = sum(terms_by_win[k][0] for k in e2e_wins)
    h2d = sum(16 * n for _, n, _ in e2e_wins)
    d2h = NP + 64 + 24 * det.cfg.max_boxes
    results = {}
    for name, fn in (("pipelined", run_pipelined), ("serial", run_serial), ("packed", run_packed)):
        fn(wins[:2])
        barrier()
        t_start = time.perf_counter()
        fn(e2e_wins)
        barrier()
        sec, terms_e = aggregate_over_ranks((time.perf_counter() - t_start) * 1e3, e2e_terms, world, dev)
        sec *= 1e-3
        results[name] = {"value": terms_e / sec / 1e9, "unit": "Gterms/s", "ms_per_step": sec / e2e_steps * 1e3,
                         "h2d_bytes_per_step": (h2d // 2 if name == "packed" else h2d) // e2e_steps, "d2h_bytes_per_step": d2h,
                         "steps": e2e_steps}
    e2e = dict(results["pipelined"], api="ddhf_host_submit/ddhf_host_wait, 2 windows in flight")
    e2e_serial = dict(results["serial"], api="ddhf_window_host")
    e2e_packed = dict(results["packed"], api="ddhf_host_submit_packed/ddhf_host_wait, 2 windows in flight, 8-byte events "
                                             "(ddhf_event8: x, y | polarity << 15, dt from a base time; bit-identical results)")

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- HBM-bound stages: algorithmic bytes over the stage's live CUDA-event time ------------------
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        hbm_kind = "measured copy bandwidth (MEASURED_PEAKS.json)"
    except Exception:
        hbm_peak, hbm_kind = 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"
    n_ev = float(np.mean([n for _, n, _ in wins[warmup:]]))
    ing_ms = float(stage[:, 0].mean())
    ing_bytes = 20.0 * n_ev + 8.0 * prm["width"] * prm["height"]          # 16 B read + 4 B written per event, 8 B per pixel
    roofline_stages = {
        "ingest": {"bound": "hbm", "kernels": "k_init, k_tile_sort, k_bucket_sort, k_worklist",
                   "achieved": ing_bytes / (ing_ms * 1e-3) / 1e9,
                   "peak": hbm_peak, "unit": "GB/s", "frac": ing_bytes / (ing_ms * 1e-3) / 1e9 / hbm_peak,
                   "algorithmic_bytes": ing_bytes, "ms": ing_ms, "peak_kind": hbm_kind,
                   "traffic": traffic_of(("k_init", "k_tile_sort", "k_bucket_sort", "k_worklist"), args.workload),
                   "traffic_source": "sum of dram__bytes_read.sum + dram__bytes_write.sum of the ingest kernels, one launch each "
                                     "(profiles/r2_traffic.csv)",
                   "note": "events are read once (16 B), bucket-sorted 4-byte items written and read once, csr_ev written; "
                           "both sort kernels are bound by shared-memory bandwidth and latency, not by HBM"},
    }

    # ---- roofline of the dominant kernel (k_ndft_score), measured live ----------------------------
    ndft_ms = float(stage[:, 1].mean())
    terms_per_step = st["terms_total"] / len(wins[warmup:])
    achieved = terms_per_step * FLOP_PER_TERM / (ndft_ms * 1e-3) / 1e12
    probe = binding.ddhf_fma_peak_probe(20.0)
    roofline = {"bound": "alu", "kernel": "k_ndft_score", "achieved": achieved, "peak": NOMINAL_FP32_TFLOPS,
                "unit": "TFLOP/s", "frac": achieved / NOMINAL_FP32_TFLOPS,
                "traffic": traffic_of(("k_ndft_score",), args.workload) if not args.spectra else None,
                "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture of this build "
                                  "(profiles/r2_traffic.csv), per launch",
                "peak_kind": "nominal FP32 FMA: 148 SM x 128 lanes x 2 flop x 1.965 GHz (DESIGN.md section 5)",
                "flop_per_term": FLOP_PER_TERM, "kernel_ms": ndft_ms,
                "gterms_per_s_kernel": terms_per_step / (ndft_ms * 1e-3) / 1e9,
                "measured_fma_peak_tflops": {"ffma": probe[0], "ffma2": probe[1]},
                "frac_of_measured_fma_peak": achieved / max(probe)}
    if args.nufft is not None:
        # the long rows went through k_nufft_score and did not execute their terms: no roofline claim for this run
        roofline.update(achieved=None, frac=None, frac_of_measured_fma_peak=None, gterms_per_s_kernel=None,
                        note="--nufft: the terms of the direct sum are nominal for the rows the NUFFT path took")
    line = {
        "metric": "ndft_gterms_per_s", "value": rec["value"], "unit": "Gterms/s", "n_gpus": world,
        "steps": steps, "warmup": warmup, "ms_per_step": rec["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": rec["config"], "latency_ms": rec["latency_ms"],
        "clocks": rec["clocks"], "e2e": e2e, "e2e_serial": e2e_serial, "e2e_packed": e2e_packed, "gpu_launches": rec["gpu_launches"],
        "roofline": roofline, "roofline_stages": roofline_stages,
        "paper_context": "DDHF 2.39 ms/frame, YOLOv11-n 12.40 ms/frame on an NVIDIA L40-8Q, 33.3 ms windows (PAPER.md L154-156)",
    }
    det.close()
    del h_ev, h_ev8, hbufs, st
    torch.cuda.empty_cache()

    # ---- the variants of SURVEY.md section 8(d), each with its own clocks ------------------------------
    if world == 1 and not args.no_sub and args.workload == "cfg4":
        from paper_2603_08386_b200 import workloads
        sub = {}
        sub_steps = min(steps, 10)

        def run_sub(key, wl_, **kw):
            r, s_ = measure(wl_, steps=kw.pop("steps", sub_steps), warmup=3, dev=dev, local_rank=local_rank, name=key, **kw)
            s_["det"].close()
            del s_
            torch.cuda.empty_cache()
            sub[key] = r

        run_sub("cfg4_score_all", w, score_all=True)
        run_sub("cfg4_table2_thresholds", w, params=dict(w.params, tau_sf=0.89, tau_comb=1.5))
        run_sub("cfg4_spectra_to_hbm", w, spectra=True)
        # long rows by the NUFFT path; reported apart -- its Gterms/s is nominal
        for m in (32, 64, 128):
            run_sub(f"cfg4_nufft_rows_ge_{m}", w, nufft=m)
        run_sub("cfg4_nufft_score_all", w, nufft=64, score_all=True)
        run_sub("paper_point", workloads.paper_native())
        run_sub("cfg3", workloads.make(3))
        w5 = workloads.make(5, n_windows=100)
        run_sub("cfg5_stream_100_windows", w5, steps=100)
        run_sub("cfg5_stream_100_windows_slide", w5, steps=100, slide=True)
        line["sub"] = sub

    if not args.no_cpu_baseline:
        full = args.workload in ("cfg4", "cfg3", "paper")
        r = time_oracle(w, 1, 0, crop=(w.width, w.height) if full else (640, 360))      # cfg4: ~27 s on 16 cores
        line["cpu_baseline"] = {"value": r["value"], "unit": "Gterms/s", "cores": r["cores"], "kind": "oracle",
                                "sample": r["sample"], "ms": r["ms_per_step"]}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
