"""Helpers shared by the GPU parity tests: run the CUDA path through the C ABI binding and
compare it with the float64 oracle, stage by stage.

Tolerances (north_star):
  CSR                 bit-exact
  power               |P_gpu - P_oracle| <= 1e-3 * max_j P_oracle  per pixel
  SF, score           relative 1e-3 (they are ratios of sums / order statistics of P)
  mask / f0 / boxes   bit-exact, except pixels whose SF or score lies within 1e-3 relative of
                      its threshold (excluded) and f0 ties (top-2 SNR within 1e-3 relative)
"""
from __future__ import annotations

import numpy as np

POWER_TOL = 1e-3
REL_TOL = 1e-3


def run_gpu(params, events, t0, window_us, *, score_all=False, want_power=True, want_debug=False,
            max_active=None, max_boxes=4096, max_events=None, timing=False, max_scored=0, **det_kw):
    from paper_2603_08386_b200 import binding
    det = binding.Detector(params, max_events=max_events or max(len(events), 1),
                           max_active=max_active, max_boxes=max_boxes, max_scored=max_scored, score_all=score_all,
                           want_power=want_power, want_debug=want_debug, timing=timing, **det_kw)
    d_ev = det.upload(events) if len(events) else None
    det.window(d_ev, len(events), t0, window_us)
    res = det.results()
    if timing:
        res["stage_ms"] = det.stage_ms()
    res["launches"] = binding.ddhf_launches_per_window(det.h)
    res["merge_alpha"] = float(params.get("merge_alpha", 0.0))
    det.close()
    return res


def check_csr(gpu, orc):
    assert gpu["n_in"] == orc["n_in"], (gpu["n_in"], orc["n_in"])
    assert gpu["n_dropped"] == orc["n_dropped"]
    assert np.array_equal(gpu["row_ptr"], orc["row_ptr"]), "row_ptr differs"
    assert np.array_equal(gpu["csr_ev"], orc["csr_ev"]), "csr_ev differs"
    assert gpu["n_active"] == orc["n_active"]
    assert np.array_equal(gpu["active_idx"], orc["active_idx"]), "active_idx differs"


def power_error(gpu_power, orc_power, counts=None):
    """max over pixels of max_j |P_gpu - P_orc| / (peak_orc + 2e-4 n^2), to be compared with POWER_TOL,
    i.e. |dP| <= 1e-3 peak + 2e-7 n^2 (n = events of the pixel; `counts`, else the floor below).
    The first term is north_star's bound.  The second is the FP32 floor of a direct sum: each of the
    n terms of X carries ~1e-7 of rounding, so |dP| <= 2 |X| |dX| can reach 2e-7 n^2 whatever the
    peak is -- it only matters for pixels whose events cancel almost everywhere (an ON and an OFF
    event 1 us apart have a peak power of 1e-5 against sum|w|^2 = 2).  Without `counts` the
    denominator is floored at 1e-6 (powers are in units of w^2 = 1)."""
    if len(orc_power) == 0:
        return 0.0
    peak = orc_power.max(axis=1)
    den = np.maximum(peak, 1e-6)
    if counts is not None:
        den = den + 2e-4 * np.asarray(counts, dtype=np.float64)[: len(peak)] ** 2
    err = np.abs(gpu_power.astype(np.float64) - orc_power).max(axis=1) / den
    return float(err.max())


def active_counts(orc):
    """events per active pixel, in active_idx order"""
    return np.diff(orc["row_ptr"])[orc["active_idx"]]


def near(value, thr, rel=REL_TOL):
    return np.abs(value - thr) <= rel * abs(thr)


#: filled by check_maps: how many pixels the last call left out of the exact comparisons
last_counts: dict = {}


def check_maps(gpu, orc, params, *, score_all, oracle_mod=None, orc_power=None, allow_ill=False,
               max_ill=None, power_of=None):
    """SF, score, f0_idx and mask on all pixels.  Returns the boolean map of pixels that are
    within tolerance of a threshold (excluded from the exact comparisons).

    By default (`allow_ill=False`) EVERY active pixel's SF and every scored pixel's score is held to
    1e-3 against the oracle.  `allow_ill=True` (randomised and edge-case streams with one- and two-event
    pixels) leaves out "ill-conditioned" pixels (R30: spectrum at the FP32 floor of the direct
    sum); `max_ill` bounds their number (asserted).  `last_counts` records how many active pixels were
    left out: "ill" and "edge" (within 1e-3 relative of a threshold, north_star).  `power_of(pix)`
    returns the oracle spectrum of one pixel on demand (full-size runs without a stored spectrum): it is
    used to settle f0 ties."""
    act = np.zeros(gpu["sf"].size, bool)
    act[orc["active_idx"]] = True
    act = act.reshape(gpu["sf"].shape)
    # inactive pixels
    assert np.isnan(gpu["sf"][~act]).all()
    assert (gpu["score"][~act] == 0).all() and (gpu["f0_idx"][~act] == -1).all()
    assert (gpu["mask"][~act] == 0).all()
    # SF.  (a) The SF stage itself: the GPU's SF against eq. 7 evaluated in float64 on the GPU's own
    # spectrum.  (b) Against the oracle's SF at REL_TOL -- except on ill-conditioned pixels: SF takes
    # the logarithm of every bin, and a bin whose power is below what the power tolerance resolves
    # (exact nulls of a two-event pixel, a balanced DC bin: the oracle has 1e-28 there, FP32 leaves
    # 1e-12) moves log P by O(1).  A pixel is ill-conditioned when the first-order bound
    # mean_k min(1, 2e-6 peak / P_k) of that effect exceeds 3e-4; such pixels are only held to (a).
    sf_g, sf_o = gpu["sf"][act].astype(np.float64), orc["sf"][act]
    sf_err = np.abs(sf_g - sf_o) / np.maximum(np.abs(sf_o), 1e-30)
    ill_map = np.zeros_like(act)
    if allow_ill and orc_power is not None and len(orc_power) == len(orc["active_idx"]) and len(orc_power):
        k_lo, eps = params["k_lo"], params["sf_eps"]
        Pt = np.maximum(orc_power[:, k_lo:], eps)
        cond = np.minimum(1.0, 2e-6 * orc_power.max(axis=1)[:, None] / Pt).mean(axis=1)
        # ... and a pixel whose whole spectrum lies below the FP32 floor of the sum (events that cancel)
        ill = (cond > 3e-4) | (orc_power.max(axis=1) <= 2e-6 * active_counts(orc)[: len(orc_power)].astype(np.float64) ** 2)
        ill_map.ravel()[orc["active_idx"][ill]] = True
        sf_err[ill_map[act]] = 0.0
    if orc_power is not None and "power" in gpu and len(gpu["power"]) == len(orc_power) == len(orc["active_idx"]) and len(orc_power):
        Pg = np.maximum(gpu["power"].astype(np.float64)[:, params["k_lo"]:], params["sf_eps"])
        sf_from_gpu = np.exp(np.log(Pg).mean(axis=1)) / Pg.mean(axis=1)
        stage_err = np.abs(gpu["sf"].ravel()[orc["active_idx"]].astype(np.float64) - sf_from_gpu) / sf_from_gpu
        assert stage_err.max(initial=0) <= 5e-5, f"SF stage rel err {stage_err.max()}"
    assert sf_err.max(initial=0) <= REL_TOL, f"SF rel err {sf_err.max()}"
    n_ill = int(ill_map.sum())
    if max_ill is not None:
        assert n_ill <= max_ill, f"{n_ill} ill-conditioned pixels (FP32 floor, DESIGN.md R30), allowed {max_ill}"
    edge_sf = (near(orc["sf"], params["tau_sf"]) | (ill_map & near(orc["sf"], params["tau_sf"], rel=0.05))) & act
    # score is evaluated where score_all or SF <= tau_sf
    scored_o = act & (np.ones_like(act) if score_all else (orc["sf"] <= params["tau_sf"]))
    cmp_px = scored_o & ~edge_sf & ~ill_map          # ill-conditioned pixels: a median or a window maximum near 0
    assert np.isfinite(gpu["score"]).all() and (gpu["score"] >= 0).all()
    s_g, s_o = gpu["score"][cmp_px].astype(np.float64), orc["score"][cmp_px]
    # strict: relative to the oracle's score (north_star).  With allow_ill (R31): an absolute
    # floor of 1e-3 is added -- a pixel whose events cancel exactly scores 0 in the oracle and ~1e-4
    # (rounding noise over sf_eps) on the GPU; scores are compared with tau_comb >= 1
    s_err = np.abs(s_g - s_o) / (np.abs(s_o) + (1.0 if allow_ill else 1e-30))
    s_err[(s_g == 0) & (s_o == 0)] = 0.0
    assert s_err.max(initial=0) <= REL_TOL, f"score err {s_err.max()} at {np.argmax(s_err)}"
    if not score_all:
        skipped = act & ~scored_o & ~edge_sf
        assert (gpu["score"][skipped] == 0).all() and (gpu["f0_idx"][skipped] == -1).all()
    # f0 index: equal unless the oracle's two best candidates tie within tolerance
    diff = cmp_px & (gpu["f0_idx"] != orc["f0_idx"])
    n_tie = int(diff.sum())
    if diff.any():
        assert oracle_mod is not None and (orc_power is not None or power_of is not None), \
            f"{diff.sum()} f0_idx mismatches and no spectra to check ties"
        row_of = {int(p): r for r, p in enumerate(orc["active_idx"])}
        W = gpu["sf"].shape[1]
        for y, x in zip(*np.nonzero(diff)):
            r = row_of[int(y) * W + int(x)]
            if orc_power is not None:
                if r >= len(orc_power):
                    continue
                P = orc_power[r]
            else:
                P = power_of(int(y) * W + int(x))
            _, _, snr, _, _ = oracle_mod.comb_score(P, params)
            g, o = gpu["f0_idx"][y, x], orc["f0_idx"][y, x]
            assert g >= 0 and abs(snr[g] - snr[o]) <= REL_TOL * snr[o], \
                f"f0_idx {g} vs {o} at ({x},{y}): snr {snr[g]} vs {snr[o]}"
    # mask
    edge = edge_sf | (near(orc["score"], params["tau_comb"]) & scored_o)
    bad = (gpu["mask"] != orc["mask"]) & ~edge
    assert not bad.any(), f"{bad.sum()} mask mismatches outside tolerance"
    last_counts.clear()
    last_counts.update(active=int(act.sum()), ill=n_ill, edge=int((edge & act).sum()), f0_ties=n_tie,
                       compared_sf=int(act.sum()) - n_ill, compared_score=int(cmp_px.sum()),
                       mask_equal=bool(np.array_equal(gpu["mask"], orc["mask"])),
                       sf_err=float(sf_err.max(initial=0)), score_err=float(s_err.max(initial=0)))
    return edge


def check_merged_boxes(gpu, oracle_mod, alpha):
    """Eq. 12 detections vs the oracle's merge of the GPU's own boxes (exact: same expression in
    double precision on both sides)."""
    if "merged_boxes" not in gpu:
        return
    import numpy as _np
    want = oracle_mod.merge_boxes(gpu["boxes"], float(_np.float32(alpha)))
    got = gpu["merged_boxes"]
    assert len(got) == len(want), (len(got), len(want))
    for k in ("x0", "y0", "x1", "y1", "n_pix", "label"):
        assert _np.array_equal(got[k], want[k]), f"merged_boxes.{k} differ"


def check_boxes_against_oracle_ccl(gpu, oracle_mod, a_min, max_boxes=4096):
    """GPU CCL/boxes vs the oracle's CCL run on the GPU's own mask (exact)."""
    labels, boxes, total = oracle_mod.ccl_boxes(gpu["mask"], a_min, max_boxes=max_boxes)
    if "labels" in gpu:
        assert np.array_equal(gpu["labels"], labels), "labels differ"
    assert gpu["n_boxes_total"] == total and gpu["n_boxes"] == len(boxes)
    for k in ("x0", "y0", "x1", "y1", "n_pix", "label"):
        assert np.array_equal(gpu["boxes"][k], boxes[k]), f"boxes.{k} differ"
    if gpu.get("merge_alpha", 0) > 0:
        check_merged_boxes(gpu, oracle_mod, gpu["merge_alpha"])
