"""GPU edge cases of the C ABI: empty and degenerate inputs, capacity limits, error codes,
determinism, the host-buffer (end-to-end) entry point."""
import ctypes as C

import numpy as np
import pytest

from paper_2603_08386_b200 import workloads as wl

import gpu_util as gu

pytestmark = pytest.mark.gpu

SMALL = dict(wl.preset(1), width=48, height=40)


def test_empty_window(oracle):
    ev = np.zeros(0, dtype=wl.EVENT_DTYPE)
    gpu = gu.run_gpu(SMALL, ev, 0, 20_000)
    assert gpu["n_in"] == 0 and gpu["n_active"] == 0 and gpu["n_boxes"] == 0
    assert (gpu["row_ptr"] == 0).all() and gpu["mask"].sum() == 0 and np.isnan(gpu["sf"]).all()


def test_all_events_dropped(oracle):
    ev = wl.random_window(3, 48, 40, 1000, 20_000)
    ev["t"] += 1_000_000                      # all after the window
    gpu = gu.run_gpu(SMALL, ev, 0, 20_000)
    assert gpu["n_in"] == 0 and gpu["n_dropped"] == 1000 and gpu["n_active"] == 0


def test_unsorted_input_and_bad_coordinates(oracle):
    ev = wl.random_window(4, 48, 40, 20_000, 20_000, hot_fraction=0.3, out_of_range=0.15,
                          time_sorted=False)
    prm = dict(SMALL, n_min=2)
    orc = oracle.window(prm, ev, 0, 20_000, score_all=True)
    gpu = gu.run_gpu(prm, ev, 0, 20_000, score_all=True)
    gu.check_csr(gpu, orc)
    assert gpu["n_dropped"] > 1000
    assert gu.power_error(gpu["power"], orc["power"]) <= gu.POWER_TOL
    gu.check_maps(gpu, orc, prm, score_all=True, oracle_mod=oracle, orc_power=orc["power"])


def test_nonzero_t0_and_negative_times(oracle):
    ev = wl.random_window(5, 48, 40, 8000, 30_000)
    ev["t"] -= 10_000                          # stream spans [-10 ms, 20 ms)
    prm = dict(SMALL, n_min=2)
    for t0 in (-10_000, -3_333, 5_000):
        orc = oracle.window(prm, ev, t0, 15_000, score_all=True)
        gpu = gu.run_gpu(prm, ev, t0, 15_000, score_all=True)
        gu.check_csr(gpu, orc)
        assert gu.power_error(gpu["power"], orc["power"]) <= gu.POWER_TOL


def test_single_hot_pixel_long_row(oracle):
    """All events on one pixel: one very long row (row sort, chunk loop, size class > 8)."""
    n = 6000
    rng = np.random.default_rng(7)
    ev = np.zeros(n, dtype=wl.EVENT_DTYPE)
    ev["x"], ev["y"] = 5, 7
    ev["t"] = np.sort(rng.integers(0, 20_000, size=n))
    ev["p"] = rng.integers(0, 2, size=n) * 2 - 1
    orc = oracle.window(SMALL, ev, 0, 20_000, score_all=True)
    gpu = gu.run_gpu(SMALL, ev, 0, 20_000, score_all=True)
    gu.check_csr(gpu, orc)
    assert gpu["n_active"] == 1
    assert gu.power_error(gpu["power"], orc["power"]) <= gu.POWER_TOL
    gu.check_maps(gpu, orc, SMALL, score_all=True, oracle_mod=oracle, orc_power=orc["power"])


def test_single_event_pixels_flat_spectrum(oracle):
    """n_min = 1: one-event pixels have P = w^2 = 1 in every bin (massive ties in the median)."""
    ev = wl.random_window(8, 48, 40, 600, 20_000)
    prm = dict(SMALL, n_min=1)
    orc = oracle.window(prm, ev, 0, 20_000, score_all=True)
    gpu = gu.run_gpu(prm, ev, 0, 20_000, score_all=True)
    gu.check_csr(gpu, orc)
    single = np.flatnonzero(np.diff(orc["row_ptr"])[orc["active_idx"]] == 1)
    assert len(single) > 100
    assert np.allclose(gpu["power"][single], 1.0, atol=1e-5)
    assert np.allclose(gpu["sf"].ravel()[orc["active_idx"][single]], 1.0, atol=1e-5)
    assert np.allclose(gpu["score"].ravel()[orc["active_idx"][single]], 1.0, atol=1e-4)
    gu.check_maps(gpu, orc, prm, score_all=True, oracle_mod=oracle, orc_power=orc["power"])


@pytest.mark.parametrize("nf,klo,fmin", [(8, 0, 50.0), (33, 1, 0.0), (256, 0, 12.5), (257, 1, 0.0),
                                         (512, 2, 0.0), (513, 1, 3.0), (1025, 1, 0.0), (2048, 0, 1.0)])
def test_grid_shapes(oracle, nf, klo, fmin):
    """Ragged n_freq (not a multiple of 32), every kernel instantiation, k_lo and f_min != 0."""
    ev = wl.random_window(9 + nf, 32, 24, 4000, 20_000, hot_fraction=0.2)
    df = 2000.0 / nf
    prm = dict(SMALL, width=32, height=24, n_freq=nf, df_hz=df, k_lo=klo, f_min_hz=fmin, n_min=3,
               f0_min_hz=max(100.0, 12 * df), f0_step_hz=10.0, n_f0=40 if nf > 64 else 3,
               n_harm=4 if nf > 64 else 1, h_min=2 if nf > 64 else 1,
               half_bw_bins=2 if nf > 64 else 0)
    orc = oracle.window(prm, ev, 0, 20_000, score_all=True)
    gpu = gu.run_gpu(prm, ev, 0, 20_000, score_all=True)
    gu.check_csr(gpu, orc)
    assert gu.power_error(gpu["power"], orc["power"]) <= gu.POWER_TOL
    gu.check_maps(gpu, orc, prm, score_all=True, oracle_mod=oracle, orc_power=orc["power"])


def test_large_sensor_2048_bin_digits(oracle):
    """2048 x 1100 pixels (21-bit pixel index): the partition runs with 2048-bin digits and the
    1-CTA-per-SM shared-memory layout; unsorted input with a hot corner and bad events."""
    W, H, T = 2048, 1100, 30_000
    ev = wl.random_window(77, W, H, 300_000, T, hot_fraction=0.3, out_of_range=0.02, time_sorted=False)
    prm = dict(SMALL, width=W, height=H, n_min=4)
    orc = oracle.window(prm, ev, 0, T)
    gpu = gu.run_gpu(prm, ev, 0, T, max_active=orc["n_active"] + 8)
    gu.check_csr(gpu, orc)
    assert gpu["n_active"] > 1000
    assert gu.power_error(gpu["power"], orc["power"]) <= gu.POWER_TOL
    gu.check_maps(gpu, orc, prm, score_all=False, oracle_mod=oracle, orc_power=orc["power"])
    gu.check_boxes_against_oracle_ccl(gpu, oracle, prm["a_min"])


def test_longest_window_keeps_phase_exact(oracle):
    """window_us = 2^31 - 1 (35.8 minutes): f t reaches 1e7 cycles at 5 kHz.  The 64-bit fixed-point
    phase constants keep 2^-32 turns, so the power error stays at the level of short windows
    (a float32 phase would be off by whole cycles)."""
    T = (1 << 31) - 1
    rng = np.random.default_rng(31)
    n_pix, per = 150, 24
    px = rng.choice(48 * 40, size=n_pix, replace=False)
    x = np.repeat(px % 48, per)
    y = np.repeat(px // 48, per)
    t = rng.integers(0, T, size=n_pix * per, dtype=np.int64)
    pol = rng.integers(0, 2, size=n_pix * per).astype(np.int16) * 2 - 1
    ev = np.zeros(n_pix * per, dtype=wl.EVENT_DTYPE)
    ev["x"], ev["y"], ev["p"], ev["t"] = x, y, pol, t
    ev = ev[np.argsort(ev["t"], kind="stable")]
    prm = dict(wl.preset(4), width=48, height=40, n_min=6)
    orc = oracle.window(prm, ev, 0, T)
    gpu = gu.run_gpu(prm, ev, 0, T)
    gu.check_csr(gpu, orc)
    assert gpu["n_active"] == n_pix
    err = gu.power_error(gpu["power"], orc["power"])
    assert err <= 2e-5, err
    gu.check_maps(gpu, orc, prm, score_all=False, oracle_mod=oracle, orc_power=orc["power"])


def test_capacity_truncation(oracle):
    w = wl.make(1)
    prm = dict(w.params, n_min=1, a_min=1, tau_sf=2.0, tau_comb=0.0)    # every active pixel is a detection
    orc = oracle.window(prm, w.events, 0, w.window_us, score_all=True, max_boxes=1 << 16)
    gpu = gu.run_gpu(prm, w.events, 0, w.window_us, score_all=True, max_active=100, max_boxes=5)
    assert gpu["overflow"] == 3
    assert gpu["n_active"] == orc["n_active"] > 100
    assert np.array_equal(gpu["active_idx"], orc["active_idx"][:100])        # lowest indices kept
    assert gu.power_error(gpu["power"], orc["power"][:100]) <= gu.POWER_TOL
    # per-pixel maps stay complete even though the compact outputs are truncated
    gu.check_maps(gpu, orc, prm, score_all=True, oracle_mod=oracle, orc_power=orc["power"])
    assert gpu["n_boxes"] == 5 and gpu["n_boxes_total"] == orc["n_boxes_total"]
    assert np.array_equal(gpu["boxes"]["label"], orc["boxes"]["label"][:5])


def test_error_codes():
    from paper_2603_08386_b200 import binding
    bad = [dict(n_freq=4), dict(n_freq=4096), dict(df_hz=0.0), dict(n_f0=0), dict(n_harm=17),
           dict(k_lo=-1), dict(width=0), dict(sf_eps=0.0),
           # harmonic windows that exclude more bins than the band sorter holds
           dict(n_freq=2048, df_hz=1.0, n_harm=16, half_bw_bins=40, h_min=1, f0_min_hz=100.0)]
    for b in bad:
        with pytest.raises(binding.DdhfError) as e:
            binding.ddhf_create(binding.make_config(dict(SMALL, **b), max_events=10))
        assert e.value.code == binding.DDHF_E_INVAL, b
    det = binding.Detector(SMALL, max_events=10)
    ev = det.upload(wl.random_window(1, 48, 40, 20, 20_000))
    with pytest.raises(binding.DdhfError) as e:
        det.window(ev, 20, 0, 20_000)
    assert e.value.code == binding.DDHF_E_CAPACITY
    with pytest.raises(binding.DdhfError) as e:
        det.window(ev, 10, 0, 0)
    assert e.value.code == binding.DDHF_E_INVAL
    with pytest.raises(binding.DdhfError) as e:
        det.window(ev, 10, 0, 1 << 31)
    assert e.value.code == binding.DDHF_E_INVAL
    det.close()


def test_deterministic_and_stateless():
    """Two runs (with another window in between) give bit-identical outputs."""
    w = wl.make(2)
    from paper_2603_08386_b200 import binding
    det = binding.Detector(w.params, max_events=len(w.events), want_power=True)
    d_ev = det.upload(w.events)
    det.window(d_ev, len(w.events), 0, w.window_us)
    a = det.results()
    det.window(d_ev, len(w.events) // 2, 0, w.window_us // 2)
    det.results()
    det.window(d_ev, len(w.events), 0, w.window_us)
    b = det.results()
    det.close()
    for k in ("row_ptr", "csr_ev", "active_idx", "power", "sf", "score", "f0_idx", "mask", "labels", "boxes"):
        same = (np.array_equal(a[k], b[k], equal_nan=True) if a[k].dtype.kind == "f"
                else np.array_equal(a[k], b[k]))
        assert same, k


@pytest.mark.parametrize("score_all", [False, True])
def test_scoring_queue_overflow_scores_in_place(score_all):
    """A deferred-scoring queue of 3 rows: every further pixel is scored inside the NDFT kernel.
    Both paths run the same code on the same float spectrum, so all outputs are bit-identical
    to those of a queue that holds every pixel."""
    w = wl.make(2)
    prm = dict(w.params, n_min=3)
    a = gu.run_gpu(prm, w.events, 0, w.window_us, score_all=score_all, want_debug=True)
    b = gu.run_gpu(prm, w.events, 0, w.window_us, score_all=score_all, want_debug=True, max_scored=3)
    assert a["n_scored"] == b["n_scored"] and a["n_scored"] > 3
    for k in ("sf", "score", "f0_idx", "mask", "labels", "boxes", "comb_debug"):
        same = (np.array_equal(a[k], b[k], equal_nan=True) if a[k].dtype.kind == "f"
                else np.array_equal(a[k], b[k]))
        assert same, k


def test_host_buffer_entry_point_matches_device_path():
    """ddhf_window_host (H2D + kernels + D2H inside the call) == ddhf_window on device buffers."""
    import torch
    from paper_2603_08386_b200 import binding
    w = wl.make(2)
    ref = gu.run_gpu(w.params, w.events, 0, w.window_us, want_power=True)
    cfg = binding.make_config(w.params, max_events=len(w.events), flags=binding.DDHF_FLAG_TIMING)
    h = binding.ddhf_create(cfg)
    NP = w.width * w.height
    ev = torch.from_numpy(np.ascontiguousarray(w.events).view(np.uint8).copy()).pin_memory()
    host = dict(
        row_ptr=np.zeros(NP + 1, np.int32), csr_ev=np.zeros(len(w.events), np.uint32),
        active_idx=np.zeros(NP, np.int32), power=np.zeros((NP, cfg.n_freq), np.float32),
        sf=np.zeros(NP, np.float32), score=np.zeros(NP, np.float32), f0_idx=np.zeros(NP, np.int32),
        mask=np.zeros(NP, np.uint8), labels=np.zeros(NP, np.int32),
        boxes=np.zeros(cfg.max_boxes, binding.BOX_DTYPE), counters=np.zeros(16, np.int32))
    out = binding.DdhfHostOutputs()
    for k, v in host.items():
        setattr(out, k, v.ctypes.data)
    for _ in range(2):                       # second call reuses the handle's buffers
        binding.ddhf_window_host(h, ev.data_ptr(), len(w.events), 0, w.window_us, out, 0)
    ms = binding.ddhf_stage_ms(h)
    assert len(ms) == 5 and all(m >= 0 for m in ms) and abs(ms[4] - sum(ms[:4])) < 0.05 * ms[4] + 0.01
    assert binding.ddhf_launches_per_window(h) >= 10
    binding.ddhf_destroy(h)
    n_in, n_act, n_box = (int(host["counters"][i]) for i in (0, 2, 3))
    assert n_in == ref["n_in"] and n_act == ref["n_active"] and n_box == ref["n_boxes"]
    assert np.array_equal(host["row_ptr"], ref["row_ptr"])
    assert np.array_equal(host["csr_ev"][:n_in], ref["csr_ev"])
    assert np.array_equal(host["active_idx"][:n_act], ref["active_idx"])
    assert np.array_equal(host["power"][:n_act], ref["power"])
    assert np.array_equal(host["mask"].reshape(ref["mask"].shape), ref["mask"])
    assert np.array_equal(host["score"].reshape(ref["mask"].shape), ref["score"])
    assert np.array_equal(host["labels"].reshape(ref["mask"].shape), ref["labels"])
    assert np.array_equal(host["boxes"][:n_box], ref["boxes"])


def test_pipelined_host_submit_wait_matches_device_path():
    """ddhf_host_submit / ddhf_host_wait: two windows in flight on two buffer sets, different
    windows back to back; every window's outputs equal the device-buffer path; error codes."""
    import torch
    from paper_2603_08386_b200 import binding
    w = wl.make(5, n_windows=4)
    wins = [w.window_slice(k) for k in range(4)]
    refs = [gu.run_gpu(w.params, w.events[lo:lo + n], t0, w.window_us, max_events=len(w.events))
            for lo, n, t0 in wins]
    cfg = binding.make_config(w.params, max_events=len(w.events))
    h = binding.ddhf_create(cfg)
    NP = w.width * w.height
    ev = torch.from_numpy(np.ascontiguousarray(w.events).view(np.uint8).copy()).pin_memory()
    st = torch.cuda.current_stream().cuda_stream
    bufs, outs = [], []
    for _ in range(2):
        t = dict(mask=torch.zeros(NP, dtype=torch.uint8).pin_memory(),
                 score=torch.zeros(NP, dtype=torch.float32).pin_memory(),
                 labels=torch.zeros(NP, dtype=torch.int32).pin_memory(),
                 boxes=torch.zeros(cfg.max_boxes * 6, dtype=torch.int32).pin_memory(),
                 counters=torch.zeros(16, dtype=torch.int32).pin_memory())
        o = binding.DdhfHostOutputs()
        for k, v in t.items():
            setattr(o, k, v.data_ptr())
        bufs.append(t)
        outs.append(o)
    with pytest.raises(binding.DdhfError):
        binding.ddhf_host_wait(h)                                   # nothing in flight

    def check(k):
        t, ref = bufs[k & 1], refs[k]
        cnt = t["counters"].numpy()
        assert int(cnt[0]) == ref["n_in"] and int(cnt[2]) == ref["n_active"] and int(cnt[3]) == ref["n_boxes"]
        assert np.array_equal(t["mask"].numpy().reshape(ref["mask"].shape), ref["mask"])
        assert np.array_equal(t["score"].numpy().reshape(ref["mask"].shape), ref["score"])
        assert np.array_equal(t["labels"].numpy().reshape(ref["mask"].shape), ref["labels"])
        nb = ref["n_boxes"]
        assert np.array_equal(t["boxes"].numpy()[: nb * 6].view(binding.BOX_DTYPE).reshape(-1), ref["boxes"])

    for k, (lo, n, t0) in enumerate(wins):
        binding.ddhf_host_submit(h, ev.data_ptr() + 16 * lo, n, t0, w.window_us, outs[k & 1], st)
        if k == 1:
            with pytest.raises(binding.DdhfError):                  # a third window in flight
                binding.ddhf_host_submit(h, ev.data_ptr(), wins[0][1], 0, w.window_us, outs[0], st)
        if k >= 1:
            binding.ddhf_host_wait(h)
            check(k - 1)
    binding.ddhf_host_wait(h)
    check(len(wins) - 1)
    bad = binding.DdhfHostOutputs()
    bad.csr_ev = bufs[0]["mask"].data_ptr()
    with pytest.raises(binding.DdhfError):
        binding.ddhf_host_submit(h, ev.data_ptr(), wins[0][1], 0, w.window_us, bad, st)
    binding.ddhf_destroy(h)


def test_fma_probe_reports_plausible_peak():
    from paper_2603_08386_b200 import binding
    scalar, packed = binding.ddhf_fma_peak_probe(5.0)
    print(f"FMA probe: scalar {scalar:.1f} TFLOP/s, packed {packed:.1f} TFLOP/s")
    assert 20.0 < max(scalar, packed) < 90.0


@pytest.mark.parametrize("alpha", [0.6, 1.5, 19.05])
def test_box_merge_many_boxes(oracle, alpha):
    """Eq. 12 on a few hundred boxes: a lenient threshold setting turns every active noise pixel
    cluster into a box; merged detections must equal the oracle's merge of the same boxes."""
    w = wl.make(2)
    prm = dict(w.params, n_min=2, tau_sf=0.99, tau_comb=0.5, a_min=1, merge_alpha=alpha)
    gpu = gu.run_gpu(prm, w.events, 0, w.window_us)
    assert gpu["n_boxes"] > 100
    gu.check_merged_boxes(gpu, oracle, alpha)
    assert 1 <= len(gpu["merged_boxes"]) <= gpu["n_boxes"]
    if alpha > 10:
        assert len(gpu["merged_boxes"]) < gpu["n_boxes"]


def test_box_merge_disabled_leaves_output_alone(oracle):
    w = wl.make(1)
    prm = dict(w.params, merge_alpha=0.0)
    gpu = gu.run_gpu(prm, w.events, 0, w.window_us)
    assert "merged_boxes" not in gpu and int(gpu["counters"][8]) == 0


@pytest.mark.parametrize("n_hot", [4096, 4097, 8200, 30_000])
def test_split_row_segments(oracle, n_hot):
    """A row longer than 4096 events is split into segments of <= 1024 events whose partial sums are
    combined along a fixed tree (ndft.cu): 4096 stays whole, 4097 gives 5 segments (one tree level),
    8200 gives 9 (two levels), 30 000 gives 30.  Everything is compared with the oracle."""
    rng = np.random.default_rng(n_hot)
    bg = wl.random_window(21, 48, 40, 6000, 20_000, hot_fraction=0.2)
    hot = np.zeros(n_hot, dtype=wl.EVENT_DTYPE)
    hot["x"], hot["y"] = 17, 23
    hot["t"] = rng.integers(0, 20_000, size=n_hot)
    # a rotor at 300 Hz, duty 0.3: ON at the start of the pulse, OFF at its end, plus noise
    k = np.arange(n_hot)
    hot["t"][::2] = ((k[::2] // 2 % 6) * 3333 + rng.integers(0, 40, size=len(k[::2]))) % 20_000
    hot["p"] = np.where(k % 2 == 0, 1, -1)
    ev = np.concatenate([bg, hot])
    ev = ev[np.argsort(ev["t"], kind="stable")]
    prm = dict(SMALL, n_min=3)
    orc = oracle.window(prm, ev, 0, 20_000, score_all=True)
    gpu = gu.run_gpu(prm, ev, 0, 20_000, score_all=True)
    gu.check_csr(gpu, orc)
    assert np.diff(orc["row_ptr"]).max() >= n_hot
    assert gu.power_error(gpu["power"], orc["power"]) <= gu.POWER_TOL
    gu.check_maps(gpu, orc, prm, score_all=True, oracle_mod=oracle, orc_power=orc["power"])
    # the split is deterministic: a second run gives the same bits
    gpu2 = gu.run_gpu(prm, ev, 0, 20_000, score_all=True)
    assert np.array_equal(gpu["power"], gpu2["power"]) and np.array_equal(gpu["score"], gpu2["score"], equal_nan=True)


@pytest.mark.slow
def test_stuck_pixel_million_events_on_config2(oracle):
    """One pixel firing 10^6 events in the window on top of the config-2 scene (PAPER.md L141 assumes
    "tens of events per pixel"): its spectrum matches the oracle, every other pixel is what it is
    without the stuck pixel, and the NDFT stage stays within 2x of (terms / the config-4 rate)."""
    w = wl.make(2)
    prm = dict(w.params, n_min=6)
    n_hot = 1_000_000
    rng = np.random.default_rng(99)
    hot = np.zeros(n_hot, dtype=wl.EVENT_DTYPE)
    hot["x"], hot["y"] = 301, 17
    hot["t"] = np.sort(rng.integers(0, w.window_us, size=n_hot)) + w.t0_us
    hot["p"] = rng.integers(0, 2, size=n_hot) * 2 - 1
    ev = np.concatenate([w.events, hot])
    ev = ev[np.argsort(ev["t"], kind="stable")]
    base = gu.run_gpu(prm, w.events, w.t0_us, w.window_us)
    gpu = gu.run_gpu(prm, ev, w.t0_us, w.window_us, timing=True)
    pix = 17 * w.width + 301
    assert gpu["counters"][9] >= 1                                         # the pixel's bucket went the giant way
    # the stuck pixel against the oracle's direct sum on its row (one pixel: seconds on one core)
    row_ptr, csr, _ = oracle.bucket(ev, w.width, w.height, w.t0_us, w.window_us)
    assert np.array_equal(gpu["row_ptr"], row_ptr) and np.array_equal(gpu["csr_ev"], csr)
    row = csr[row_ptr[pix]:row_ptr[pix + 1]]
    assert len(row) >= n_hot
    p_orc = oracle.ndft_power(row >> 1, np.where(row & 1, 1.0, -1.0), prm["f_min_hz"], prm["df_hz"], prm["n_freq"])
    r = int(np.flatnonzero(gpu["active_idx"] == pix)[0])
    err = np.abs(gpu["power"][r] - p_orc).max() / p_orc.max()
    print(f"stuck pixel: {len(row)} events, power err / peak {err:.2e}, stage ms {gpu['stage_ms']}")
    assert err <= gu.POWER_TOL
    sf_o = oracle.spectral_flatness(p_orc, prm["k_lo"], prm["sf_eps"])
    assert abs(gpu["sf"].ravel()[pix] - sf_o) <= 1e-3 * sf_o
    # every other pixel: exactly the maps of the scene without the stuck pixel
    other = np.ones(w.width * w.height, dtype=bool)
    other[pix] = False
    for k in ("sf", "score", "f0_idx"):
        assert np.array_equal(gpu[k].ravel()[other], base[k].ravel()[other], equal_nan=True), k
    m_g, m_b = gpu["mask"].ravel().copy(), base["mask"].ravel().copy()
    assert np.array_equal(m_g[other], m_b[other])
    if m_g[pix] == m_b[pix]:
        assert np.array_equal(gpu["boxes"], base["boxes"])
    # time: terms of the window / 10 Tterms/s (the NDFT kernel's rate on config 4), within 2x
    cnt = np.diff(row_ptr)
    terms = prm["n_freq"] * float(cnt[cnt >= prm["n_min"]].sum())
    budget_ms = 2.0 * terms / 10.0e12 * 1e3
    assert gpu["stage_ms"][1] <= budget_ms, (gpu["stage_ms"], budget_ms)


@pytest.mark.parametrize("t_base_off", [0, -7_000, 3_000])
def test_packed_events_bit_identical(oracle, t_base_off):
    """8-byte events (ddhf_event8: y | polarity << 15, dt from a base time): every output equals the
    16-byte call bit for bit, and the CSR equals the oracle's; events before t_base cannot be expressed,
    so the base is at or before the first event; bad coordinates and out-of-window times included."""
    from paper_2603_08386_b200 import binding
    ev = wl.random_window(41, 48, 40, 25_000, 30_000, hot_fraction=0.3, out_of_range=0.1, time_sorted=False)
    ev["t"] += 10_000
    t_base = int(ev["t"].min()) + min(t_base_off, 0)
    t0 = 12_000 + max(t_base_off, 0)
    prm = dict(SMALL, n_min=2)
    ref = gu.run_gpu(prm, ev, t0, 20_000, score_all=True)
    ev8 = wl.pack_events(ev, t_base)
    det = binding.Detector(prm, max_events=len(ev), score_all=True, want_power=True)
    d8 = det.torch.from_numpy(ev8.view(np.uint8).copy()).to(det.device)
    det.window_packed(d8, len(ev8), t_base, t0, 20_000)
    got = det.results()
    det.close()
    row_ptr, csr, dropped = oracle.bucket(ev, 48, 40, t0, 20_000)
    assert np.array_equal(got["row_ptr"], row_ptr) and np.array_equal(got["csr_ev"], csr) and got["n_dropped"] == dropped
    for k in ("row_ptr", "csr_ev", "active_idx", "power", "sf", "score", "f0_idx", "mask", "boxes"):
        same = (np.array_equal(got[k], ref[k], equal_nan=True) if got[k].dtype.kind == "f" else np.array_equal(got[k], ref[k]))
        assert same, k


@pytest.mark.parametrize("window_us", [50_000, (1 << 31) - 1])
def test_giant_buckets_sorted_by_helper_ctas(oracle, window_us):
    """Buckets of more than 65 536 events are cut into chunks of whole tiles and sorted by helper CTAs
    (ingest.cu, "giant buckets"): two stuck pixels in different buckets, one bucket with two hot pixels and a
    background, input not time-sorted, with 4-byte and (window 2^31 - 1 us) 8-byte items.  CSR bit-exact."""
    W, H = 346, 260
    rng = np.random.default_rng(window_us % 1000)
    parts = [wl.random_window(5, W, H, 150_000, 50_000, hot_fraction=0.1)]
    for (x, y, n) in ((10, 3, 300_000), (200, 200, 120_000), (40, 100, 90_000), (41, 100, 70_000)):
        e = np.zeros(n, dtype=wl.EVENT_DTYPE)
        e["x"], e["y"] = x, y
        e["t"] = rng.integers(0, 50_000, size=n)
        e["p"] = rng.integers(0, 2, size=n) * 2 - 1
        parts.append(e)
    ev = np.concatenate(parts)
    ev = ev[rng.permutation(len(ev))]
    prm = dict(wl.preset(2), n_min=6)
    gpu = gu.run_gpu(prm, ev, 0, window_us, want_power=False)
    row_ptr, csr, dropped = oracle.bucket(ev, W, H, 0, window_us)
    assert gpu["counters"][9] >= 3, gpu["counters"]                     # DDHF_CNT_N_GIANT
    assert gpu["n_dropped"] == dropped and gpu["n_in"] == len(csr)
    assert np.array_equal(gpu["row_ptr"], row_ptr) and np.array_equal(gpu["csr_ev"], csr)
    cnt = np.diff(row_ptr)
    assert gpu["n_active"] == int((cnt >= 6).sum())


@pytest.mark.parametrize("n_harm,d,max_scored", [(12, 12, 0), (12, 12, 50), (16, 15, 0), (16, 27, 0)])
def test_wide_harmonic_windows_use_the_larger_band_sorters(oracle, n_harm, d, max_scored):
    """Unions of harmonic windows of 300 / 496 / 880 of 2048 bins: the rank band of the complement medians needs the
    512- and 1024-value band sorters (the BASELINE configs need 256).  Every active pixel scored, per-candidate values
    compared; with a queue of 50 rows the 512-value variant also scores in place inside the NDFT kernel."""
    W, H, T = 40, 24, 100_000
    w1 = wl.make(1)
    ev = wl.random_window(77, W, H, 25_000, T, hot_fraction=0.3)
    # a periodic source on a few pixels so that some spectra have real harmonic structure
    rng = np.random.default_rng(8)
    tt = np.round(np.arange(0, T, 1e6 / 210.0)).astype(np.int64)
    per = wl._pack(np.repeat([5, 6, 7], len(tt)), np.full(3 * len(tt), 9), np.ones(3 * len(tt), int), np.tile(tt, 3))
    ev = np.concatenate([ev, per])
    ev = ev[np.argsort(ev["t"], kind="stable")]
    prm = dict(w1.params, width=W, height=H, f_min_hz=0.0, df_hz=5000.0 / 2048, n_freq=2048, k_lo=1, n_harm=n_harm,
               half_bw_bins=d, h_min=4, n_min=4, f0_min_hz=100.0, f0_step_hz=2.5, n_f0=80, tau_sf=0.9, tau_comb=1.5, a_min=1)
    orc = oracle.window(prm, ev, 0, T, score_all=True, want_power=True)
    gpu = gu.run_gpu(prm, ev, 0, T, score_all=True, want_power=True, want_debug=True, max_scored=max_scored)
    gu.check_csr(gpu, orc)
    assert gpu["n_scored"] == orc["n_active"] > 400
    assert gu.power_error(gpu["power"], orc["power"]) <= gu.POWER_TOL
    gu.check_maps(gpu, orc, prm, score_all=True, oracle_mod=oracle, orc_power=orc["power"])
    worst = 0.0
    for r in range(0, gpu["n_active"], 7):
        s, fi, snr, num, med = oracle.comb_score(orc["power"][r], prm)
        dd = gpu["comb_debug"][r].astype(np.float64)
        for k, ref in enumerate((snr, num, med)):
            e = np.abs(dd[:, k] - ref) / np.maximum(np.abs(ref), 1e-30)
            e[(ref == 0) & (dd[:, k] == 0)] = 0
            worst = max(worst, e.max())
    assert worst <= gu.REL_TOL, worst
    print(f"H={n_harm} d={d} queue={max_scored or 'all'}: per-candidate worst rel err {worst:.2e}, {gu.last_counts}")
