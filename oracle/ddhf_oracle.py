"""ctypes/numpy face of the float64 CPU oracle (oracle/ddhf_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Nothing under paper_2603_08386_b200/ imports it
and it imports nothing from there.  Argument marshalling only -- every number comes from
the C functions, which are the paper's definitions written out (see ddhf_oracle.h).
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)
sys.path.pop(0)


class OrcConfig(C.Structure):
    _fields_ = [
        ("width", C.c_int32), ("height", C.c_int32),
        ("f_min_hz", C.c_double), ("df_hz", C.c_double), ("n_freq", C.c_int32),
        ("f0_min_hz", C.c_double), ("f0_step_hz", C.c_double), ("n_f0", C.c_int32),
        ("n_harm", C.c_int32), ("half_bw_bins", C.c_int32), ("h_min", C.c_int32),
        ("n_min", C.c_int32), ("a_min", C.c_int32),
        ("tau_sf", C.c_double), ("tau_comb", C.c_double), ("sf_eps", C.c_double),
        ("k_lo", C.c_int32), ("score_all", C.c_int32),
    ]


ORC_EVENT = np.dtype([("x", "<u2"), ("y", "<u2"), ("p", "<i2"), ("pad", "<u2"), ("t", "<i8")],
                     align=True)
ORC_BOX = np.dtype([("x0", "<i4"), ("y0", "<i4"), ("x1", "<i4"), ("y1", "<i4"),
                    ("n_pix", "<i4"), ("label", "<i4")])

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp = C.c_void_p
        L.orc_bucket.restype = C.c_int64
        L.orc_bucket.argtypes = [vp, C.c_int64, C.c_int32, C.c_int32, C.c_int64, C.c_int64, vp, vp]
        L.orc_ndft_power.restype = None
        L.orc_ndft_power.argtypes = [vp, vp, C.c_int64, C.c_double, C.c_double, C.c_int32, vp]
        L.orc_spectral_flatness.restype = C.c_double
        L.orc_spectral_flatness.argtypes = [vp, C.c_int32, C.c_int32, C.c_double]
        L.orc_comb_score.restype = C.c_double
        L.orc_comb_score.argtypes = [vp, C.POINTER(OrcConfig), C.POINTER(C.c_int32), vp, vp, vp]
        L.orc_merge_boxes.restype = C.c_int32
        L.orc_merge_boxes.argtypes = [vp, C.c_int32, C.c_double, vp]
        L.orc_ccl_boxes.restype = C.c_int32
        L.orc_ccl_boxes.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, vp, vp, C.c_int32,
                                    C.POINTER(C.c_int32)]
        L.orc_window.restype = C.c_int
        L.orc_window.argtypes = [C.POINTER(OrcConfig), vp, C.c_int64, C.c_int64, C.c_int64,
                                 vp, vp, vp, vp, C.c_int64, vp, vp, vp, vp, vp, vp, C.c_int32, vp]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def make_config(params: dict, score_all: bool = False) -> OrcConfig:
    c = OrcConfig()
    for name, _ in OrcConfig._fields_:
        if name == "score_all":
            c.score_all = int(score_all)
        else:
            setattr(c, name, params[name])
    return c


def num_threads() -> int:
    return int(lib().orc_num_threads())


def bucket(events: np.ndarray, width: int, height: int, t0_us: int, window_us: int):
    ev = np.ascontiguousarray(events, dtype=ORC_EVENT)
    n = len(ev)
    row_ptr = np.zeros(width * height + 1, dtype=np.int32)
    csr = np.zeros(max(n, 1), dtype=np.uint32)
    dropped = lib().orc_bucket(_p(ev), n, width, height, t0_us, window_us, _p(row_ptr), _p(csr))
    return row_ptr, csr[: row_ptr[-1]], int(dropped)


def ndft_power(t_us, w, f_min_hz: float, df_hz: float, n_freq: int) -> np.ndarray:
    t = np.ascontiguousarray(t_us, dtype=np.int64)
    ww = np.ascontiguousarray(w, dtype=np.float64)
    assert t.shape == ww.shape
    out = np.zeros(n_freq, dtype=np.float64)
    lib().orc_ndft_power(_p(t), _p(ww), len(t), f_min_hz, df_hz, n_freq, _p(out))
    return out


def spectral_flatness(power, k_lo: int, eps: float) -> float:
    pw = np.ascontiguousarray(power, dtype=np.float64)
    return float(lib().orc_spectral_flatness(_p(pw), len(pw), k_lo, eps))


def comb_score(power, params: dict):
    """Returns (score, f0_idx, snr[n_f0], numerator[n_f0], median[n_f0])."""
    pw = np.ascontiguousarray(power, dtype=np.float64)
    cfg = make_config({**params, "n_freq": len(pw)})
    snr = np.zeros(cfg.n_f0); num = np.zeros(cfg.n_f0); med = np.zeros(cfg.n_f0)
    fi = C.c_int32(-1)
    s = lib().orc_comb_score(_p(pw), C.byref(cfg), C.byref(fi), _p(snr), _p(num), _p(med))
    return float(s), int(fi.value), snr, num, med


def ccl_boxes(mask: np.ndarray, a_min: int, max_boxes: int = 1 << 20):
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    h, w = m.shape
    labels = np.zeros((h, w), dtype=np.int32)
    boxes = np.zeros(max_boxes, dtype=ORC_BOX)
    tot = C.c_int32(0)
    nb = lib().orc_ccl_boxes(_p(m), w, h, a_min, _p(labels), _p(boxes), max_boxes, C.byref(tot))
    return labels, boxes[:nb].copy(), int(tot.value)


def merge_boxes(boxes: np.ndarray, alpha: float) -> np.ndarray:
    """Eq. 12 box merge (transitive); boxes: ORC_BOX array sorted by label."""
    b = np.ascontiguousarray(boxes, dtype=ORC_BOX)
    out = np.zeros(max(len(b), 1), dtype=ORC_BOX)
    n = lib().orc_merge_boxes(_p(b), len(b), float(alpha), _p(out))
    return out[:n]


def window(params: dict, events: np.ndarray, t0_us: int, window_us: int, *,
           score_all: bool = False, want_power: bool = True, max_boxes: int = 4096,
           power_rows_cap: int | None = None) -> dict:
    """Run a0-a8 on one window.  Returns a dict of numpy arrays (float64 where floating)."""
    cfg = make_config(params, score_all)
    ev = np.ascontiguousarray(events, dtype=ORC_EVENT)
    n = len(ev)
    NP = cfg.width * cfg.height
    row_ptr = np.zeros(NP + 1, dtype=np.int32)
    csr = np.zeros(max(n, 1), dtype=np.uint32)
    active = np.zeros(max(NP, 1), dtype=np.int32)
    sf = np.zeros(NP); score = np.zeros(NP)
    f0_idx = np.zeros(NP, dtype=np.int32)
    mask = np.zeros(NP, dtype=np.uint8)
    labels = np.zeros(NP, dtype=np.int32)
    boxes = np.zeros(max(max_boxes, 1), dtype=ORC_BOX)
    counters = np.zeros(5, dtype=np.int64)
    power = None
    cap = 0
    if want_power:
        # number of active pixels is not known before the call: size by a cheap count
        key = ev["y"].astype(np.int64) * cfg.width + ev["x"]
        ok = (ev["t"] >= t0_us) & (ev["t"] < t0_us + window_us) & (ev["x"] < cfg.width) & (ev["y"] < cfg.height)
        cnt = np.bincount(key[ok], minlength=NP)
        cap = int((cnt >= max(cfg.n_min, 1)).sum())
        if power_rows_cap is not None:
            cap = min(cap, power_rows_cap)
        power = np.zeros((max(cap, 1), cfg.n_freq), dtype=np.float64)
    rc = lib().orc_window(C.byref(cfg), _p(ev), n, t0_us, window_us, _p(row_ptr), _p(csr),
                          _p(active), _p(power), cap, _p(sf), _p(score), _p(f0_idx), _p(mask),
                          _p(labels), _p(boxes), max_boxes, _p(counters))
    assert rc == 0
    n_active = int(counters[2])
    H, W = cfg.height, cfg.width
    return dict(row_ptr=row_ptr, csr_ev=csr[: row_ptr[-1]], active_idx=active[:n_active],
                power=None if power is None else power[:cap], sf=sf.reshape(H, W),
                score=score.reshape(H, W), f0_idx=f0_idx.reshape(H, W),
                mask=mask.reshape(H, W), labels=labels.reshape(H, W),
                boxes=boxes[: int(counters[3])].copy(), n_in=int(counters[0]),
                n_dropped=int(counters[1]), n_active=n_active, n_boxes=int(counters[3]),
                n_boxes_total=int(counters[4]))
