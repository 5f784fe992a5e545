"""Seeded synthetic event-camera workloads (the five BASELINE.json configs).

This module only *generates inputs*: event tuples (x, y, p, t_us) laid out as the
16-byte records the C ABI takes, plus the per-config parameter presets.  It holds
none of the method's arithmetic (no NDFT, no scoring, no bucketing) and is the one
module both the CUDA path's tests/bench and the oracle's tests may import.

The paper's recordings (Prophesee EVK4-HD, 1280x720) are private, so
these streams stand in for them.  What is taken from the paper: event tuple and
polarity convention, microsecond timestamps (L55), "tens of events per
pixel per window" (L141), rotor pixels as rectangular pulse trains with duty cycle tau
whose ON/OFF edges make events (eq. 1-5), window lengths of tens of ms (L137).
The recipe per config is SURVEY.md section 8(d); it is restated in DESIGN.md.

Everything is numpy with ``default_rng([2603, 8386, cfg])``; timestamps are int64
microseconds relative to t0 = 0 and the stream is finally sorted by time, as a camera
delivers it.  A few events fall outside [0, window) (jitter at the window edges): they
exercise the drop counter of the ingest step.
"""
from __future__ import annotations

import dataclasses
from typing import Any

import numpy as np

#: numpy view of ``ddhf_event`` (include/ddhf.h): 16 bytes, little endian.
EVENT_DTYPE = np.dtype(
    [("x", "<u2"), ("y", "<u2"), ("p", "<i2"), ("pad", "<u2"), ("t", "<i8")], align=True
)
assert EVENT_DTYPE.itemsize == 16
#: ddhf_event8 of include/ddhf.h: the same tuple in 8 bytes (timestamp as an offset from a base time)
EVENT8_DTYPE = np.dtype([("x", "<u2"), ("y_p", "<u2"), ("dt", "<u4")])
assert EVENT8_DTYPE.itemsize == 8


def pack_events(ev: np.ndarray, t_base_us: int) -> np.ndarray:
    """16-byte events -> 8-byte events (a change of container, nothing of the method): y and the polarity
    bit share a word, t becomes t - t_base_us in 32 bits."""
    dt = ev["t"].astype(np.int64) - int(t_base_us)
    assert dt.min(initial=0) >= 0 and dt.max(initial=0) < (1 << 32) and ev["y"].max(initial=0) < 32768
    out = np.zeros(len(ev), dtype=EVENT8_DTYPE)
    out["x"] = ev["x"]
    out["y_p"] = ev["y"].astype(np.uint16) | ((ev["p"] > 0).astype(np.uint16) << 15)
    out["dt"] = dt.astype(np.uint32)
    return out


@dataclasses.dataclass
class Workload:
    """One synthetic window (configs 1-4) or stream (config 5)."""

    cfg: int
    events: np.ndarray            # EVENT_DTYPE, time sorted
    params: dict[str, Any]        # fields of ddhf_config (python-side names)
    t0_us: int
    window_us: int
    hop_us: int = 0               # config 5 only
    n_windows: int = 1
    truth: dict[str, Any] = dataclasses.field(default_factory=dict)

    @property
    def width(self) -> int:
        return self.params["width"]

    @property
    def height(self) -> int:
        return self.params["height"]

    def window_slice(self, w: int) -> tuple[int, int, int]:
        """(first event index, event count, t0) of sliding window ``w`` (time-sorted stream)."""
        t0 = self.t0_us + w * self.hop_us
        t = self.events["t"]
        lo = int(np.searchsorted(t, t0, side="left"))
        hi = int(np.searchsorted(t, t0 + self.window_us, side="left"))
        return lo, hi - lo, t0


# --------------------------------------------------------------------------------------
# parameter presets (SURVEY.md 8(c) readings 4, 12, 13, 22)
# --------------------------------------------------------------------------------------

def preset(cfg: int) -> dict[str, Any]:
    """ddhf_config values for BASELINE.json config ``cfg`` (1-based).

    Thresholds: the retuned operating point of PAPER.md Fig. 3 / L172 (tau_sf 0.5,
    tau_comb 6.0), n_min 6 and h_min 4 from Table 2 (L232-233), A_min 9 = the lower BO
    bound (L234).  Table 2's own finals are in ``paper_table2()``.
    """
    common = dict(h_min=4, n_min=6, a_min=9, tau_sf=0.5, tau_comb=6.0, sf_eps=1e-12, k_lo=1,
                  f_min_hz=0.0, merge_alpha=19.05)          # alpha of eq. 12: Table 2 (L235)
    if cfg == 1:
        p = dict(width=64, height=64, window_us=20_000, df_hz=10.0, n_freq=201,
                 f0_min_hz=100.0, f0_step_hz=10.0, n_f0=31, n_harm=5, half_bw_bins=5)
    elif cfg == 2:
        p = dict(width=346, height=260, window_us=50_000, df_hz=5000.0 / 1024, n_freq=1024,
                 f0_min_hz=100.0, f0_step_hz=5.0, n_f0=81, n_harm=6, half_bw_bins=5)
    elif cfg == 3:
        p = dict(width=640, height=480, window_us=100_000, df_hz=5000.0 / 2048, n_freq=2048,
                 f0_min_hz=100.0, f0_step_hz=5.0, n_f0=81, n_harm=8, half_bw_bins=10)
    elif cfg == 4:
        p = dict(width=1280, height=720, window_us=100_000, df_hz=5000.0 / 2048, n_freq=2048,
                 f0_min_hz=100.0, f0_step_hz=5.0, n_f0=81, n_harm=8, half_bw_bins=10)
    elif cfg == 5:
        p = dict(width=1280, height=720, window_us=50_000, df_hz=5000.0 / 1024, n_freq=1024,
                 f0_min_hz=100.0, f0_step_hz=5.0, n_f0=81, n_harm=6, half_bw_bins=5)
    else:
        raise ValueError(f"no such config: {cfg}")
    return {**common, **p}


def paper_table2() -> dict[str, Any]:
    """Final hyperparameters of PAPER.md Table 2 (L226-237)."""
    return dict(tau_sf=0.89, tau_comb=1.5, n_harm=4, half_bw_bins=3, h_min=4, n_min=6,
                a_min=147, alpha=19.05)


# --------------------------------------------------------------------------------------
# building blocks
# --------------------------------------------------------------------------------------

def _pack(x, y, p, t) -> np.ndarray:
    ev = np.zeros(len(t), dtype=EVENT_DTYPE)
    ev["x"] = x
    ev["y"] = y
    ev["p"] = p
    ev["t"] = t
    return ev


def _sort_by_time(ev: np.ndarray) -> np.ndarray:
    return ev[np.argsort(ev["t"], kind="stable")]


def _poisson_noise(rng, pix_x, pix_y, lam, t_lo, t_hi) -> np.ndarray:
    """Poisson(lam) events on each listed pixel, uniform times, random polarity."""
    cnt = rng.poisson(lam, size=len(pix_x))
    n = int(cnt.sum())
    x = np.repeat(pix_x, cnt)
    y = np.repeat(pix_y, cnt)
    t = rng.integers(t_lo, t_hi, size=n, dtype=np.int64)
    p = rng.integers(0, 2, size=n).astype(np.int16) * 2 - 1
    return _pack(x, y, p, t)


def _all_pixels(width, height):
    yy, xx = np.divmod(np.arange(width * height, dtype=np.int64), width)
    return xx.astype(np.uint16), yy.astype(np.uint16)


def _rotor_events(rng, px, py, f0_hz, duty, sigma_us, t_lo, t_hi) -> np.ndarray:
    """Rect pulse train at each listed pixel (eq. 1): one ON event at the start
    of each occlusion and one OFF event ``duty`` periods later, per-pixel phase offset,
    Gaussian jitter on every event."""
    period = 1e6 / f0_hz
    n_per = int(np.ceil((t_hi - t_lo) / period)) + 1
    npx = len(px)
    phase = rng.uniform(0.0, period, size=npx)
    k = np.arange(-1, n_per)
    t_on = t_lo + phase[:, None] + k[None, :] * period            # (npx, n_per+1)
    t_off = t_on + duty * period
    t = np.concatenate([t_on.ravel(), t_off.ravel()])
    t = t + rng.normal(0.0, sigma_us, size=t.shape)
    p = np.concatenate([np.ones(t_on.size, np.int16), -np.ones(t_off.size, np.int16)])
    x = np.concatenate([np.repeat(px, len(k))] * 2)
    y = np.concatenate([np.repeat(py, len(k))] * 2)
    ti = np.rint(t).astype(np.int64)
    # keep a margin of one jitter sigma outside the window so a handful of events land
    # out of range and are dropped (and counted) by the ingest step
    keep = (ti >= t_lo - int(sigma_us)) & (ti < t_hi + int(sigma_us))
    return _pack(x[keep], y[keep], p[keep], ti[keep])


def _disc(cx, cy, r, width, height):
    y0, y1 = max(0, int(cy - r) - 1), min(height - 1, int(cy + r) + 1)
    x0, x1 = max(0, int(cx - r) - 1), min(width - 1, int(cx + r) + 1)
    yy, xx = np.mgrid[y0:y1 + 1, x0:x1 + 1]
    m = (xx - cx) ** 2 + (yy - cy) ** 2 <= r * r
    return xx[m].astype(np.uint16), yy[m].astype(np.uint16)


def _drone(rng, x0, y0, size, width, height, f0_range, duty_range, sigma_us, t_lo, t_hi,
           distinct_f0=None):
    """A size x size drone: four disc blobs (rotors) at the quadrant centres, each with
    its own blade-pass frequency."""
    r = size * 0.21
    parts, info = [], []
    for q, (qx, qy) in enumerate([(0.27, 0.27), (0.73, 0.27), (0.27, 0.73), (0.73, 0.73)]):
        px, py = _disc(x0 + qx * size, y0 + qy * size, r, width, height)
        f0 = distinct_f0[q] if distinct_f0 is not None else rng.uniform(*f0_range)
        duty = rng.uniform(*duty_range)
        parts.append(_rotor_events(rng, px, py, f0, duty, sigma_us, t_lo, t_hi))
        info.append(dict(f0_hz=float(f0), duty=float(duty), px=px, py=py))
    return np.concatenate(parts), info


def _truth_mask(width, height, rotors):
    m = np.zeros((height, width), dtype=bool)
    for r in rotors:
        m[r["py"], r["px"]] = True
    return m


# --------------------------------------------------------------------------------------
# configs
# --------------------------------------------------------------------------------------

def config1(seed_extra: int = 0) -> Workload:
    """64x64, 20 ms; Poisson(0.5) noise; one 8x8 rotor patch at 200 Hz, duty 0.28,
    jitter 50 us (duty 0.28 makes harmonics 1..5 all present)."""
    prm = preset(1)
    W, H, T = prm["width"], prm["height"], prm["window_us"]
    rng = np.random.default_rng([2603, 8386, 1, seed_extra])
    ax, ay = _all_pixels(W, H)
    noise = _poisson_noise(rng, ax, ay, 0.5, 0, T)
    yy, xx = np.mgrid[24:32, 40:48]
    px, py = xx.ravel().astype(np.uint16), yy.ravel().astype(np.uint16)
    rot = _rotor_events(rng, px, py, 200.0, 0.28, 50.0, 0, T)
    ev = _sort_by_time(np.concatenate([noise, rot]))
    rotors = [dict(f0_hz=200.0, duty=0.28, px=px, py=py)]
    return Workload(1, ev, prm, 0, T, truth=dict(rotors=rotors, mask=_truth_mask(W, H, rotors)))


def config2(seed_extra: int = 0) -> Workload:
    """346x260, 50 ms; Poisson(1) noise; one 20x20 drone of four rotor blobs, each
    f0 ~ U[150, 350] Hz, duty ~ U[0.2, 0.35], jitter 30 us."""
    prm = preset(2)
    W, H, T = prm["width"], prm["height"], prm["window_us"]
    rng = np.random.default_rng([2603, 8386, 2, seed_extra])
    ax, ay = _all_pixels(W, H)
    noise = _poisson_noise(rng, ax, ay, 1.0, 0, T)
    d, rotors = _drone(rng, 150, 110, 20, W, H, (150, 350), (0.2, 0.35), 30.0, 0, T)
    ev = _sort_by_time(np.concatenate([noise, d]))
    return Workload(2, ev, prm, 0, T, truth=dict(rotors=rotors, mask=_truth_mask(W, H, rotors)))


def _rect_clutter(rng, n_rect, W, H, T, target_events):
    """Edges of translating rectangles: every pixel a leading/trailing edge crosses emits
    a short same-polarity burst at the crossing time (opposite sign on the two edges)."""
    xs, ys, ps, ts = [], [], [], []
    crossings = []
    for _ in range(n_rect):
        w = int(rng.integers(20, 200))
        h = int(rng.integers(20, 200))
        x0 = float(rng.uniform(0, W - w))
        y0 = float(rng.uniform(0, H - h))
        speed = float(rng.uniform(20.0, 200.0)) * (1 if rng.random() < 0.5 else -1)   # px/s
        horizontal = rng.random() < 0.5
        sign = 1 if rng.random() < 0.5 else -1
        travel = speed * T * 1e-6
        for edge, pol in ((0.0, sign), (float(w if horizontal else h), -sign)):
            start = (x0 if horizontal else y0) + edge
            lo, hi = sorted((start, start + travel))
            cols = np.arange(int(np.ceil(lo)), int(np.floor(hi)) + 1)
            lim = W if horizontal else H
            cols = cols[(cols >= 0) & (cols < lim)]
            if len(cols) == 0:
                continue
            t_cross = (cols - start) / speed * 1e6
            if horizontal:
                rows = np.arange(int(y0), min(H, int(y0) + h))
                cx, cy = np.meshgrid(cols, rows, indexing="ij")
            else:
                rows = np.arange(int(x0), min(W, int(x0) + w))
                cy, cx = np.meshgrid(cols, rows, indexing="ij")
            tc = np.repeat(t_cross, len(rows))
            crossings.append((cx.ravel(), cy.ravel(), tc, pol, abs(speed)))
    n_cross = sum(len(c[0]) for c in crossings)
    lam = target_events / max(n_cross, 1)
    for cx, cy, tc, pol, spd in crossings:
        cnt = rng.poisson(lam, size=len(cx))
        n = int(cnt.sum())
        dur = 1e6 / spd                                   # time the edge spends on one pixel
        t = np.repeat(tc, cnt) + rng.uniform(0.0, dur, size=n)
        xs.append(np.repeat(cx, cnt)); ys.append(np.repeat(cy, cnt))
        ps.append(np.full(n, pol, np.int16)); ts.append(np.rint(t).astype(np.int64))
    x = np.concatenate(xs); y = np.concatenate(ys); p = np.concatenate(ps); t = np.concatenate(ts)
    keep = (t >= 0) & (t < T)
    return _pack(x[keep], y[keep], p[keep], t[keep])


def config3(seed_extra: int = 0, target_events: int = 2_000_000) -> Workload:
    """640x480, 100 ms; Poisson(2) noise; 3 drones (10-40 px) with distinct f0 in
    120-400 Hz; edges of 50 translating rectangles; about 2 M events."""
    prm = preset(3)
    W, H, T = prm["width"], prm["height"], prm["window_us"]
    rng = np.random.default_rng([2603, 8386, 3, seed_extra])
    ax, ay = _all_pixels(W, H)
    noise = _poisson_noise(rng, ax, ay, 2.0, 0, T)
    parts, rotors = [noise], []
    f0s = rng.permutation(np.linspace(120.0, 400.0, 12))
    for i, (size, x0, y0) in enumerate([(40, 100, 80), (24, 420, 200), (10, 300, 380)]):
        d, info = _drone(rng, x0, y0, size, W, H, None, (0.2, 0.35), 40.0, 0, T,
                         distinct_f0=f0s[4 * i:4 * i + 4])
        parts.append(d); rotors += info
    have = sum(len(p) for p in parts)
    parts.append(_rect_clutter(rng, 50, W, H, T, max(target_events - have, 0)))
    ev = _sort_by_time(np.concatenate(parts))
    return Workload(3, ev, prm, 0, T, truth=dict(rotors=rotors, mask=_truth_mask(W, H, rotors)))


def _hot_pixels(rng, W, H, n_hot, shake_dir, amp=5):
    """Random edge texture (straight segments) dilated by the shake amplitude along the
    shake direction; the first n_hot pixels in a seeded random order are kept."""
    m = np.zeros((H, W), dtype=bool)
    dx, dy = np.cos(shake_dir), np.sin(shake_dir)
    while m.sum() < n_hot * 1.05:
        L = rng.uniform(50, 400)
        th = rng.uniform(0, np.pi)
        x0, y0 = rng.uniform(0, W), rng.uniform(0, H)
        s = np.arange(0.0, L, 0.5)
        for a in np.arange(-amp, amp + 0.5, 0.5):
            xs = np.rint(x0 + s * np.cos(th) + a * dx).astype(np.int64)
            ys = np.rint(y0 + s * np.sin(th) + a * dy).astype(np.int64)
            ok = (xs >= 0) & (xs < W) & (ys >= 0) & (ys < H)
            m[ys[ok], xs[ok]] = True
    idx = np.flatnonzero(m.ravel())
    idx = np.sort(rng.permutation(idx)[:n_hot])
    return idx


def _shake_events(rng, hot_idx, W, mean_per_pixel, t_lo, t_hi, f_shake, phi):
    """Hot-pixel events: count ~ Poisson(mean * lognormal factor) (heavy tailed), times
    drawn with density |cos(2 pi f_s t + phi)| (the shake speed), polarity = sign of the
    velocity times a per-pixel edge sign, 10 % flipped."""
    sig = 0.8
    factor = rng.lognormal(-0.5 * sig * sig, sig, size=len(hot_idx))
    cnt = rng.poisson(mean_per_pixel * factor)
    n = int(cnt.sum())
    pix = np.repeat(hot_idx, cnt)
    edge_sign = np.repeat(rng.integers(0, 2, size=len(hot_idx)) * 2 - 1, cnt)
    t = np.empty(n, dtype=np.float64)
    todo = np.arange(n)
    w = 2 * np.pi * f_shake * 1e-6
    while len(todo):
        cand = rng.uniform(t_lo, t_hi, size=len(todo))
        acc = rng.random(len(todo)) < np.abs(np.cos(w * cand + phi))
        t[todo[acc]] = cand[acc]
        todo = todo[~acc]
    vel = np.sign(np.cos(w * t + phi))
    vel[vel == 0] = 1
    p = (vel * edge_sign).astype(np.int16)
    flip = rng.random(n) < 0.10
    p[flip] = -p[flip]
    ti = np.minimum(np.floor(t).astype(np.int64), t_hi - 1)
    return _pack((pix % W).astype(np.uint16), (pix // W).astype(np.uint16), p, ti)


def _scene4(rng, W, H, t_lo, t_hi, hot_mean, cold_mean):
    n_hot = int(round(0.05 * W * H))
    shake_dir = rng.uniform(0, np.pi)
    f_shake = rng.uniform(2.0, 8.0)
    phi = rng.uniform(0, 2 * np.pi)
    hot = _hot_pixels(rng, W, H, n_hot, shake_dir)
    cold_mask = np.ones(W * H, dtype=bool)
    cold_mask[hot] = False
    cold = np.flatnonzero(cold_mask)
    ev_hot = _shake_events(rng, hot, W, hot_mean, t_lo, t_hi, f_shake, phi)
    ev_cold = _poisson_noise(rng, (cold % W).astype(np.uint16), (cold // W).astype(np.uint16),
                             cold_mean, t_lo, t_hi)
    return ev_hot, ev_cold, dict(f_shake_hz=float(f_shake), n_hot=n_hot)


def config4(seed_extra: int = 0, scale: float = 1.0) -> Workload:
    """1280x720, 100 ms, about 10 M events: 5 % of the pixels (shaken edge texture) hold
    60 % of the events with a heavy tail; Poisson(4.57) elsewhere; two drones.
    ``scale`` < 1 shrinks the sensor (both sides) for tests; rates are unchanged."""
    prm = preset(4)
    if scale != 1.0:
        prm["width"] = max(64, int(prm["width"] * scale))
        prm["height"] = max(64, int(prm["height"] * scale))
    W, H, T = prm["width"], prm["height"], prm["window_us"]
    rng = np.random.default_rng([2603, 8386, 4, seed_extra])
    ev_hot, ev_cold, info = _scene4(rng, W, H, 0, T, hot_mean=130.2, cold_mean=4.57)
    parts, rotors = [ev_hot, ev_cold], []
    for size, fx, fy in [(36, 0.25, 0.3), (24, 0.7, 0.6)]:
        size = min(size, W // 3, H // 3)
        d, r = _drone(rng, int(fx * W), int(fy * H), size, W, H, (150, 350), (0.2, 0.35), 50.0, 0, T)
        parts.append(d); rotors += r
    ev = _sort_by_time(np.concatenate(parts))
    return Workload(4, ev, prm, 0, T,
                    truth=dict(rotors=rotors, mask=_truth_mask(W, H, rotors), **info))


def config5(seed_extra: int = 0, n_windows: int = 100, scale: float = 1.0) -> Workload:
    """Streaming: the config-4 scene extended in time at 50 Mev/s, sliding windows of
    50 ms with a 10 ms hop; one drone moving at 30 px/s whose f0 sweeps 180 -> 260 Hz
    over the stream (ON events at integer crossings of the integral of f, OFF events a
    duty fraction of a period later)."""
    prm = preset(5)
    if scale != 1.0:
        prm["width"] = max(64, int(prm["width"] * scale))
        prm["height"] = max(64, int(prm["height"] * scale))
    W, H, T = prm["width"], prm["height"], prm["window_us"]
    hop = 10_000
    dur = T + (n_windows - 1) * hop
    rng = np.random.default_rng([2603, 8386, 5, seed_extra])
    # rates per 50 ms window: hot pixels 32.5, others 1.14  (-> 50 Mev/s at full size)
    k = dur / T
    ev_hot, ev_cold, info = _scene4(rng, W, H, 0, dur, hot_mean=32.5 * k, cold_mean=1.14 * k)
    # moving drone with a linear chirp
    size = min(30, W // 3, H // 3)
    f_a, f_b, duty, sigma = 180.0, 260.0, 0.28, 50.0
    full_dur = 50_000 + 99 * hop                       # the sweep is defined over the full stream
    rate = (f_b - f_a) / (full_dur * 1e-6)             # Hz per second
    parts, rotors = [ev_hot, ev_cold], []
    x_start, y_start = 0.3 * W, 0.4 * H
    r = size * 0.21
    for qx, qy in [(0.27, 0.27), (0.73, 0.27), (0.27, 0.73), (0.73, 0.73)]:
        ox, oy = _disc(qx * size, qy * size, r, 1 << 15, 1 << 15)
        npx = len(ox)
        ph0 = rng.uniform(0, 1, size=npx)
        n_cyc = int(np.ceil((f_a + f_b) / 2 * dur * 1e-6 * 1.3)) + 2
        kk = np.arange(n_cyc)
        # integral of f: f_a t + rate t^2 / 2 = k + ph0  ->  t
        target = kk[None, :] + ph0[:, None]
        t_on = (-f_a + np.sqrt(f_a * f_a + 2 * rate * target)) / rate
        f_inst = f_a + rate * t_on
        t_off = t_on + duty / f_inst
        tt = np.concatenate([t_on.ravel(), t_off.ravel()]) * 1e6
        tt = tt + rng.normal(0.0, sigma, size=tt.shape)
        pp = np.concatenate([np.ones(t_on.size, np.int16), -np.ones(t_on.size, np.int16)])
        bx = np.concatenate([np.repeat(ox, n_cyc)] * 2).astype(np.float64)
        by = np.concatenate([np.repeat(oy, n_cyc)] * 2).astype(np.float64)
        xx = np.floor(x_start + bx + 30.0 * tt * 1e-6).astype(np.int64)
        yy = np.floor(y_start + by).astype(np.int64)
        ti = np.rint(tt).astype(np.int64)
        keep = (ti >= 0) & (ti < dur) & (xx >= 0) & (xx < W) & (yy >= 0) & (yy < H)
        parts.append(_pack(xx[keep], yy[keep], pp[keep], ti[keep]))
    rotors.append(dict(f0_start_hz=f_a, f0_end_hz=f_b, duty=duty, x_start=x_start,
                       y_start=y_start, size=size, speed_px_s=30.0))
    ev = _sort_by_time(np.concatenate(parts))
    return Workload(5, ev, prm, 0, T, hop_us=hop, n_windows=n_windows,
                    truth=dict(rotors=rotors, **info))


def paper_native(seed_extra: int = 0) -> Workload:
    """The paper's own operating point on the config-4 scene: the first 33.3 ms
    of the 1280x720 window (30 FPS frames), integer modes f_k = k / T (L139), i.e.
    df = 1/T = 30.03 Hz, 167 modes up to 5 kHz (the paper never states K), and the final
    hyperparameters of Table 2 (L226-237).  The recordings differ, so this is context only."""
    w = config4(seed_extra)
    T = 33_300
    ev = w.events[w.events["t"] < T + 200]
    t2 = paper_table2()
    prm = dict(w.params, window_us=T, df_hz=1e6 / T, n_freq=167, n_harm=t2["n_harm"],
               half_bw_bins=t2["half_bw_bins"], h_min=t2["h_min"], n_min=t2["n_min"], a_min=t2["a_min"],
               tau_sf=t2["tau_sf"], tau_comb=t2["tau_comb"], merge_alpha=t2["alpha"],
               f0_min_hz=100.0, f0_step_hz=5.0, n_f0=81)
    return Workload(4, ev, prm, 0, T, truth=w.truth)


def make(cfg: int, **kw) -> Workload:
    return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}[cfg](**kw)


def random_window(seed: int, width: int, height: int, n_events: int, window_us: int,
                  hot_fraction: float = 0.0, out_of_range: float = 0.0,
                  time_sorted: bool = True) -> np.ndarray:
    """Unstructured test stream: uniform pixels (optionally a hot subset), uniform times,
    random polarity, optionally a fraction of events outside the window / sensor and an
    unsorted order.  Used by the bucketing and edge-case tests."""
    rng = np.random.default_rng([2603, 8386, 99, seed])
    x = rng.integers(0, width, size=n_events)
    y = rng.integers(0, height, size=n_events)
    if hot_fraction > 0:
        hot = rng.random(n_events) < hot_fraction
        x[hot] = rng.integers(0, max(1, width // 16), size=int(hot.sum()))
        y[hot] = rng.integers(0, max(1, height // 16), size=int(hot.sum()))
    t = rng.integers(0, window_us, size=n_events, dtype=np.int64)
    p = rng.integers(0, 2, size=n_events).astype(np.int16) * 2 - 1
    if out_of_range > 0:
        bad = rng.random(n_events) < out_of_range
        kind = rng.integers(0, 4, size=n_events)
        t[bad & (kind == 0)] = -1 - rng.integers(0, 1000, size=int((bad & (kind == 0)).sum()))
        t[bad & (kind == 1)] = window_us + rng.integers(0, 1000, size=int((bad & (kind == 1)).sum()))
        x[bad & (kind == 2)] = width + rng.integers(0, 50, size=int((bad & (kind == 2)).sum()))
        y[bad & (kind == 3)] = height + rng.integers(0, 50, size=int((bad & (kind == 3)).sum()))
    ev = _pack(x, y, p, t)
    if time_sorted:
        ev = _sort_by_time(ev)
    return ev
