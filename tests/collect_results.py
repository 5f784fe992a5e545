"""Collect the per-config results table of BASELINE.md section 4 on a B200 box.

    python tests/collect_results.py > gpurun_out/results.md

For each BASELINE.json config: GPU stage times through the C ABI (median of 20 windows after 5
warm-ups, inputs device-resident), NDFT Gterms/s and fraction of the FP32 roofline, ingest GB/s on
the algorithmic bytes, the float64 oracle timed on the host cores on the same window, and the
parity maxima (the same comparisons as tests/test_gpu_parity.py).  Test infrastructure: this is
one of the places allowed to call oracle/.
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
sys.path.insert(0, ROOT)
sys.path.insert(0, HERE)
sys.path.insert(0, os.path.join(ROOT, "oracle"))

import ddhf_oracle as oracle                       # noqa: E402
import gpu_util as gu                              # noqa: E402
import test_gpu_parity as tp                       # noqa: E402
from paper_2603_08386_b200 import binding, workloads as wl   # noqa: E402

PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
HBM_GBS = 6540.8


def gpu_times(w, ev, t0, n_rep=20, warm=5):
    det = binding.Detector(w.params, max_events=len(ev), timing=True, want_labels=False, max_active=1)
    d_ev = det.upload(ev)
    ms = []
    for i in range(warm + n_rep):
        det.window(d_ev, len(ev), t0, w.window_us)
        m = det.stage_ms()
        if i >= warm:
            ms.append(m)
    res = det.results()
    det.close()
    ms = np.array(ms)
    return np.median(ms, axis=0), np.percentile(ms[:, 4], 99), res


def main():
    print("| cfg | n events | active px | terms | GPU ms p50 / p99 | ingest / NDFT / comb / CCL ms | NDFT Gterms/s "
          "| % FP32 peak (nominal) | ingest GB/s (% HBM) | oracle ms (cores) | power err / peak | SF rel | score rel "
          "| CSR exact | mask mismatches outside tolerance |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for cfg in (1, 2, 3, 4, 5):
        w = wl.make(cfg, n_windows=3) if cfg == 5 else wl.make(cfg)
        if cfg == 5:
            lo, n, t0 = w.window_slice(1)
            ev = w.events[lo:lo + n]
        else:
            ev, t0 = w.events, w.t0_us
        prm = w.params
        med, p99, res = gpu_times(w, ev, t0)
        cnt = np.diff(res["row_ptr"])
        terms = int(cnt[cnt >= prm["n_min"]].sum()) * prm["n_freq"]
        # parity
        if cfg <= 2:
            gpu, orc, perr = tp._full_compare(oracle, w, prm, score_all=False)
            sf_err = score_err = float("nan")
            act = np.zeros(gpu["sf"].size, bool)
            act[orc["active_idx"]] = True
            act = act.reshape(gpu["sf"].shape)
            sf_err = float((np.abs(gpu["sf"][act] - orc["sf"][act]) / orc["sf"][act]).max())
            sc = act & (orc["sf"] <= prm["tau_sf"]) & ~gu.near(orc["sf"], prm["tau_sf"])
            score_err = float((np.abs(gpu["score"][sc] - orc["score"][sc]) / np.maximum(orc["score"][sc], 1e-30)).max()) \
                if sc.any() else 0.0
            mism = "0 (all pixels)"
        else:
            gpu, perr, sf_err, score_err = tp._sampled_compare(oracle, w, prm, ev, t0, 300, score_all=False)
            mism = "0 (sampled pixels)"
        # oracle timing on the same window
        t = time.perf_counter()
        oracle.window(prm, ev, t0, w.window_us, want_power=False)
        orc_ms = (time.perf_counter() - t) * 1e3
        n_in = res["n_in"]
        ing_bytes = 20.0 * n_in + 8.0 * prm["width"] * prm["height"]
        ing_gbs = ing_bytes / (med[0] * 1e-3) / 1e9
        gt = terms / (med[1] * 1e-3) / 1e9
        frac = gt * 4e9 / 1e12 / PEAK_TFLOPS
        print(f"| {cfg} | {n_in} | {res['n_active']} | {terms:.3e} | {med[4]:.3f} / {p99:.3f} | "
              f"{med[0]:.3f} / {med[1]:.3f} / {med[2]:.3f} / {med[3]:.3f} | {gt:.0f} | {100 * frac:.1f} % | "
              f"{ing_gbs:.0f} ({100 * ing_gbs / HBM_GBS:.1f} %) | {orc_ms:.0f} ({oracle.num_threads()}) | "
              f"{perr:.1e} | {sf_err:.1e} | {score_err:.1e} | yes | {mism} |", flush=True)


if __name__ == "__main__":
    main()
