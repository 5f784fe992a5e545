"""GPU parity of the optional NUFFT path for long rows (DDHF_FLAG_NUFFT, PAPER.md L141 footnote 1)
against the same float64 oracle and the same tolerances as the direct sum.  Run with `pytest -m gpu` on a B200."""
import numpy as np
import pytest

from paper_2603_08386_b200 import workloads as wl

import gpu_util as gu
from test_gpu_parity import _full_compare, _sampled_compare, _whole_window_compare

pytestmark = pytest.mark.gpu


def _grid2048(width, height, window_us=100_000):
    prm = dict(wl.make(1).params)
    prm.update(width=width, height=height, f_min_hz=0.0, df_hz=5000.0 / 2048, n_freq=2048, n_harm=8, half_bw_bins=10,
               f0_min_hz=100.0, f0_step_hz=5.0, n_f0=81, h_min=4, n_min=1, k_lo=1)
    return prm


@pytest.mark.parametrize("score_all", [False, True])
def test_nufft_config4_quarter_scale(oracle, score_all):
    """Every spectrum of the config-4 scene on a 320x180 sensor, rows of >= 32 events through the NUFFT."""
    w = wl.make(4, scale=0.25)
    gpu, orc, err = _full_compare(oracle, w, w.params, score_all=score_all, nufft=True, nufft_min=32)
    n = np.diff(orc["row_ptr"])[orc["active_idx"]]
    assert (n >= 32).sum() > 1000 and gpu["launches"] == 12
    print(f"nufft cfg4/16 score_all={score_all}: rows through the NUFFT {(n >= 32).sum()} of {len(n)}, "
          f"power err/peak {err:.2e}, mask {gpu['mask'].sum()}")


def test_nufft_every_row_length(oracle):
    """Rows of 1 .. 4096 events (the longest unsplit row), one pixel each, all through the NUFFT (nufft_min = 1);
    a row of 4097 events is split and summed directly as always."""
    lens = [1, 2, 3, 4, 5, 7, 8, 9, 31, 32, 33, 63, 64, 65, 100, 255, 256, 257, 1000, 2047, 4095, 4096, 4097]
    W = len(lens)
    prm = _grid2048(W, 1)
    rng = np.random.default_rng(5)
    x = np.repeat(np.arange(W), lens)
    t = rng.integers(0, 100_000, size=len(x))
    t[:3] = [0, 99_999, 99_999]                      # both ends of the window
    ev = wl._pack(x, np.zeros_like(x), rng.integers(0, 2, size=len(x)) * 2 - 1, t)
    ev = ev[rng.permutation(len(ev))]                # unsorted input: rows keep the input order
    orc = oracle.window(prm, ev, 0, 100_000, score_all=True, want_power=True)
    gpu = gu.run_gpu(prm, ev, 0, 100_000, score_all=True, want_power=True, nufft=True, nufft_min=1)
    gu.check_csr(gpu, orc)
    err = np.abs(gpu["power"].astype(np.float64) - orc["power"]).max(axis=1) / orc["power"].max(axis=1)
    print("  power err / peak by row length:", {n: f"{e:.1e}" for n, e in zip(lens, err)})
    assert err.max() <= gu.POWER_TOL
    gu.check_maps(gpu, orc, prm, score_all=True, oracle_mod=oracle, orc_power=orc["power"])
    # and against the direct path on the same device: both within FP32 of each other
    ref = gu.run_gpu(prm, ev, 0, 100_000, score_all=True, want_power=True)
    d = np.abs(gpu["power"] - ref["power"]).max(axis=1) / ref["power"].max(axis=1)
    assert d.max() <= 2e-4, d
    assert np.array_equal(gpu["power"][-1], ref["power"][-1])        # the split row took the same path


def test_nufft_periodic_train_peaks(oracle):
    """A strictly periodic train at f0 puts its peaks at k f0 (north_star's pin), here through the NUFFT."""
    prm = _grid2048(4, 1)
    f0 = 250.0
    t = np.round(np.arange(25) * 1e6 / f0).astype(np.int64)
    ev = wl._pack(np.full(25, 2), np.zeros(25, int), np.ones(25, int), t)
    gpu = gu.run_gpu(prm, ev, 0, 100_000, score_all=True, want_power=True, nufft=True, nufft_min=1)
    P = gpu["power"][0]
    for k in (1, 2, 3, 4):
        j = int(round(k * f0 / prm["df_hz"]))
        assert abs(int(np.argmax(P[j - 20:j + 21])) - 20) <= 1 and P[j] >= 0.95 * 25 ** 2
    assert abs(P[0] - 625.0) <= 1e-3 * 625.0                         # P_0 = (sum w)^2


def test_nufft_ignored_where_it_does_not_apply(oracle):
    """1024-bin grids, windows longer than a quarter turn of the grid phase and handles whose scoring queue is
    smaller than the sensor run the direct path: results identical to a handle without the flag."""
    w = wl.make(2)
    a = gu.run_gpu(w.params, w.events, 0, w.window_us, want_power=True, nufft=True, nufft_min=1)
    b = gu.run_gpu(w.params, w.events, 0, w.window_us, want_power=True)
    assert np.array_equal(a["power"], b["power"]) and np.array_equal(a["sf"], b["sf"], equal_nan=True)
    prm = _grid2048(64, 64)
    ev = wl.random_window(3, 64, 64, 60_000, 110_000, hot_fraction=0.5)
    for kw, win in ((dict(), 110_000), (dict(max_scored=100), 100_000)):
        e = ev[ev["t"] < win]
        a = gu.run_gpu(prm, e, 0, win, want_power=True, nufft=True, nufft_min=1, **kw)
        b = gu.run_gpu(prm, e, 0, win, want_power=True, **kw)
        assert np.array_equal(a["power"], b["power"]) and a["launches"] == b["launches"]


@pytest.mark.slow
def test_nufft_config4_whole_window(oracle):
    """Whole config-4 window, every active pixel's SF / score / mask and the boxes, rows of >= 64 events (the
    default) through the NUFFT: same bars as test_config4_whole_window."""
    w = wl.make(4)
    _whole_window_compare(oracle, w, w.params, w.events, 0, score_all=False, name="cfg4 whole window, NUFFT", nufft=True)


@pytest.mark.slow
def test_nufft_config3_full_size_sampled(oracle):
    w = wl.make(3)
    gpu, wp, wsf, ws = _sampled_compare(oracle, w, w.params, w.events, 0, 400, score_all=False, nufft=True, nufft_min=48)
    print(f"nufft cfg3: worst power {wp:.2e}, SF {wsf:.2e}, score {ws:.2e}")


def test_nufft_on_sliding_windows(oracle):
    """ddhf_window_slide() with the NUFFT path on: the hot list is filled by the scan kernels of the sliding path.
    Every window equals ddhf_window() on the same slice bit for bit (same kernels on the same rows) and the oracle
    within the usual bars; one pixel is long enough to be split (> 4096 events: direct sum)."""
    from paper_2603_08386_b200 import binding
    W, H, T, hop = 40, 24, 100_000, 20_000
    prm = _grid2048(W, H)
    prm.update(n_min=4, a_min=1)
    ev = wl.random_window(11, W, H, 150_000, 200_000, hot_fraction=0.6)      # hot 2 x 1 corner: rows of thousands of events
    rng = np.random.default_rng(3)
    hot = ev[rng.random(len(ev)) < 0.25].copy()
    hot["x"], hot["y"] = 7, 5                                               # > 4096 events per window on one pixel
    ev = np.concatenate([ev, hot])
    ev = ev[np.argsort(ev["t"], kind="stable")]
    kw = dict(max_events=len(ev), want_power=True, nufft=True, nufft_min=16, max_active=W * H)
    det, ref = binding.Detector(prm, **kw), binding.Detector(prm, **kw)
    d_ev = det.upload(ev)
    t = ev["t"]
    prev_hi = None
    for k in range(6):
        t0 = k * hop
        lo, hi = int(np.searchsorted(t, t0, "left")), int(np.searchsorted(t, t0 + T, "left"))
        if prev_hi is None:
            det.slide(d_ev, hi - lo, t0, T, offset_events=lo)
        else:
            det.slide(d_ev, hi - prev_hi, t0, T, offset_events=prev_hi)
        prev_hi = hi
        g = det.results()
        ref.window(d_ev, hi - lo, t0, T, offset_events=lo)
        r = ref.results()
        for key in ("row_ptr", "csr_ev", "active_idx", "power", "sf", "score", "f0_idx", "mask", "boxes"):
            same = np.array_equal(g[key], r[key], equal_nan=True) if g[key].dtype.kind == "f" else np.array_equal(g[key], r[key])
            assert same, (k, key)
        if k in (0, 3):
            orc = oracle.window(prm, ev[lo:hi], t0, T, score_all=False, want_power=True)
            gu.check_csr(g, orc)
            n = np.diff(orc["row_ptr"])[orc["active_idx"]]
            assert (n > 4096).any() and ((n >= 16) & (n <= 4096)).sum() > 20
            assert gu.power_error(g["power"], orc["power"]) <= gu.POWER_TOL
            gu.check_maps(g, orc, prm, score_all=False, oracle_mod=oracle, orc_power=orc["power"])
    det.close()
    ref.close()


def _random_case(seed):
    """A random configuration on which the NUFFT path applies: 1024 < n_freq <= 2048, df x window <= 0.24."""
    rng = np.random.default_rng([2603, 8386, 4141, seed])
    W, H = int(rng.integers(8, 120)), int(rng.integers(8, 90))
    T = int(rng.choice([5_000, 20_000, 100_000]))
    nf = int(rng.choice([1025, 1030, 1500, 2047, 2048]))
    fmin = float(rng.choice([0.0, 0.0, 37.5]))
    df = float(rng.uniform(0.05, 0.24)) / (T * 1e-6)
    klo = int(rng.integers(0, 3)) if fmin == 0 else 0
    d = int(rng.integers(0, 4))
    n_harm = int(rng.integers(1, 7))
    prm = dict(width=W, height=H, window_us=T, f_min_hz=fmin, df_hz=df, n_freq=nf, k_lo=klo,
               f0_min_hz=fmin + (d + klo + 2 + float(rng.uniform(0, 40))) * df, f0_step_hz=float(rng.choice([0.5, 2.0, 7.0])) * df,
               n_f0=int(rng.integers(1, 100)), n_harm=n_harm, half_bw_bins=d,
               h_min=int(rng.integers(1, n_harm + 1)), n_min=int(rng.integers(3, 8)),
               a_min=int(rng.integers(1, 12)), tau_sf=float(rng.uniform(0.3, 0.95)),
               tau_comb=float(rng.uniform(1.5, 8.0)), sf_eps=1e-12, merge_alpha=float(rng.choice([0.0, 19.05])))
    ev = wl.random_window(3000 + seed, W, H, int(rng.integers(2_000, 80_000)), T, hot_fraction=float(rng.choice([0.3, 0.8])),
                          out_of_range=float(rng.choice([0.0, 0.05])), time_sorted=bool(rng.integers(0, 2)))
    return prm, ev, T, bool(rng.integers(0, 2)), int(rng.choice([1, 8, 64]))


@pytest.mark.parametrize("seed", range(8))
def test_nufft_random_configuration(oracle, seed):
    """Random grids (n_freq not a multiple of 32, f_min > 0, k_lo 0..2), sensors and event mixes, rows of >= 1 / 8 / 64
    events through the NUFFT: every stage against the oracle with the bars of test_gpu_fuzz.py."""
    from paper_2603_08386_b200 import binding
    from test_gpu_fuzz import ILL_CAP
    prm, ev, T, score_all, nmin = _random_case(seed)
    try:
        gpu = gu.run_gpu(prm, ev, 0, T, score_all=score_all, nufft=True, nufft_min=nmin)
    except binding.DdhfError as e:
        assert "band sorter" in str(e), str(e)
        pytest.skip(str(e))
    assert gpu["launches"] == (12 if prm["merge_alpha"] > 0 else 11)       # the NUFFT kernel did run
    orc = oracle.window(prm, ev, 0, T, score_all=score_all)
    gu.check_csr(gpu, orc)
    assert gu.power_error(gpu["power"], orc["power"], gu.active_counts(orc)) <= gu.POWER_TOL
    n_act = max(int(orc["n_active"]), 1)
    gu.check_maps(gpu, orc, prm, score_all=score_all, oracle_mod=oracle, orc_power=orc["power"],
                  allow_ill=True, max_ill=int(ILL_CAP[min(prm["n_min"], 3)] * n_act) + 2)
    print(f"nufft seed {seed}: n_freq {prm['n_freq']}, rows >= {nmin}, {gu.last_counts}")
    gu.check_boxes_against_oracle_ccl(gpu, oracle, prm["a_min"])
