"""Thin Python face of the C ABI in include/ddhf.h (ctypes; argument marshalling only).

Every step of the hot path runs in the CUDA kernels of ``libddhf.so``; torch is used here
for device memory and streams only.  There is no CPU fallback: if the shared library is
missing or fails to load, importing a symbol from it raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Any

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("DDHF_LIB", os.path.join(_HERE, "libddhf.so"))

DDHF_OK, DDHF_E_INVAL, DDHF_E_CAPACITY, DDHF_E_CUDA, DDHF_E_NOMEM = 0, -1, -2, -3, -4
DDHF_FLAG_SCORE_ALL, DDHF_FLAG_TIMING, DDHF_FLAG_NUFFT = 1, 2, 4
(CNT_N_IN, CNT_N_DROPPED, CNT_N_ACTIVE, CNT_N_BOXES, CNT_N_BOXES_TOTAL, CNT_OVERFLOW,
 CNT_N_SCORED, CNT_N_COMPONENTS, CNT_N_MERGED) = range(9)
N_COUNTERS = 16

#: every symbol include/ddhf.h declares
EXPORTS = ["ddhf_create", "ddhf_workspace_bytes", "ddhf_window", "ddhf_window_packed", "ddhf_window_slide", "ddhf_slide_reset",
           "ddhf_host_submit_packed",
           "ddhf_window_host",
           "ddhf_host_submit", "ddhf_host_wait",
           "ddhf_stage_ms", "ddhf_launches_per_window", "ddhf_fma_peak_probe", "ddhf_destroy",
           "ddhf_last_error", "ddhf_version",
           "ddhf_boxes_noalloc_setup", "ddhf_boxes_noalloc", "ddhf_boxes_noalloc_error"]

BOX_DTYPE = np.dtype([("x0", "<i4"), ("y0", "<i4"), ("x1", "<i4"), ("y1", "<i4"),
                      ("n_pix", "<i4"), ("label", "<i4")])


class DdhfConfig(C.Structure):
    _fields_ = [
        ("width", C.c_int32), ("height", C.c_int32),
        ("f_min_hz", C.c_double), ("df_hz", C.c_double), ("n_freq", C.c_int32),
        ("f0_min_hz", C.c_double), ("f0_step_hz", C.c_double), ("n_f0", C.c_int32),
        ("n_harm", C.c_int32), ("half_bw_bins", C.c_int32), ("h_min", C.c_int32),
        ("n_min", C.c_int32), ("a_min", C.c_int32), ("merge_alpha", C.c_float),
        ("tau_sf", C.c_float), ("tau_comb", C.c_float), ("sf_eps", C.c_float),
        ("k_lo", C.c_int32),
        ("max_events", C.c_int64), ("max_active", C.c_int32), ("max_boxes", C.c_int32),
        ("max_scored", C.c_int32),
        ("flags", C.c_uint32),
    ]


class DdhfOutputs(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in
                ("row_ptr", "csr_ev", "active_idx", "power", "sf", "score", "f0_idx", "mask",
                 "labels", "boxes", "counters", "merged_boxes", "comb_debug")]


class DdhfHostOutputs(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in
                ("row_ptr", "csr_ev", "active_idx", "power", "sf", "score", "f0_idx", "mask",
                 "labels", "boxes", "counters", "merged_boxes")]


_lib = None


def lib() -> C.CDLL:
    """Load libddhf.so (built by paper_2603_08386_b200/build.py).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} not found: build it with `python -m paper_2603_08386_b200.build` "
                "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.ddhf_create.restype = C.c_int
        L.ddhf_create.argtypes = [C.POINTER(DdhfConfig), C.POINTER(vp)]
        L.ddhf_workspace_bytes.restype = C.c_size_t
        L.ddhf_workspace_bytes.argtypes = [vp]
        L.ddhf_window.restype = C.c_int
        L.ddhf_window.argtypes = [vp, vp, C.c_int64, C.c_int64, C.c_int64, vp,
                                  C.POINTER(DdhfOutputs), vp]
        L.ddhf_window_packed.restype = C.c_int
        L.ddhf_window_packed.argtypes = [vp, vp, C.c_int64, C.c_int64, C.c_int64, C.c_int64, vp,
                                         C.POINTER(DdhfOutputs), vp]
        L.ddhf_host_submit_packed.restype = C.c_int
        L.ddhf_host_submit_packed.argtypes = [vp, vp, C.c_int64, C.c_int64, C.c_int64, C.c_int64,
                                              C.POINTER(DdhfHostOutputs), vp]
        L.ddhf_window_slide.restype = C.c_int
        L.ddhf_window_slide.argtypes = [vp, vp, C.c_int64, C.c_int64, C.c_int64, vp,
                                        C.POINTER(DdhfOutputs), vp]
        L.ddhf_slide_reset.restype = C.c_int
        L.ddhf_slide_reset.argtypes = [vp]
        L.ddhf_window_host.restype = C.c_int
        L.ddhf_window_host.argtypes = [vp, vp, C.c_int64, C.c_int64, C.c_int64,
                                       C.POINTER(DdhfHostOutputs), vp]
        L.ddhf_host_submit.restype = C.c_int
        L.ddhf_host_submit.argtypes = [vp, vp, C.c_int64, C.c_int64, C.c_int64,
                                       C.POINTER(DdhfHostOutputs), vp]
        L.ddhf_host_wait.restype = C.c_int
        L.ddhf_host_wait.argtypes = [vp]
        L.ddhf_stage_ms.restype = C.c_int
        L.ddhf_stage_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.ddhf_launches_per_window.restype = C.c_int
        L.ddhf_launches_per_window.argtypes = [vp]
        L.ddhf_fma_peak_probe.restype = C.c_int
        L.ddhf_fma_peak_probe.argtypes = [C.c_float, C.POINTER(C.c_float), vp]
        L.ddhf_destroy.restype = C.c_int
        L.ddhf_destroy.argtypes = [vp]
        L.ddhf_boxes_noalloc_setup.restype = C.c_int
        L.ddhf_boxes_noalloc_setup.argtypes = []
        L.ddhf_boxes_noalloc.restype = C.c_int
        L.ddhf_boxes_noalloc.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_float, C.c_int32, vp, vp, vp, vp, vp]
        L.ddhf_boxes_noalloc_error.restype = C.c_char_p
        L.ddhf_boxes_noalloc_error.argtypes = []
        L.ddhf_last_error.restype = C.c_char_p
        L.ddhf_last_error.argtypes = [vp]
        L.ddhf_version.restype = C.c_char_p
        L.ddhf_version.argtypes = []
        _lib = L
    return _lib


class DdhfError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"ddhf error {code}: {msg}")
        self.code = code


def make_config(params: dict[str, Any], *, max_events: int, max_active: int | None = None,
                max_boxes: int = 4096, max_scored: int = 0, flags: int = 0) -> DdhfConfig:
    c = DdhfConfig()
    for name in ("width", "height", "f_min_hz", "df_hz", "n_freq", "f0_min_hz", "f0_step_hz",
                 "n_f0", "n_harm", "half_bw_bins", "h_min", "n_min", "a_min", "tau_sf", "tau_comb",
                 "sf_eps", "k_lo"):
        setattr(c, name, params[name])
    c.merge_alpha = float(params.get("merge_alpha", 0.0))
    c.max_events = int(max_events)
    c.max_active = int(max_active if max_active is not None else params["width"] * params["height"])
    c.max_boxes = int(max_boxes)
    c.max_scored = int(max_scored)
    c.flags = int(flags)
    return c


# ----------------------------------------------------------------------------------------
# the ABI calls, same names
# ----------------------------------------------------------------------------------------
def ddhf_create(cfg: DdhfConfig) -> C.c_void_p:
    h = C.c_void_p()
    rc = lib().ddhf_create(C.byref(cfg), C.byref(h))
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(None) or b"").decode())
    return h


def ddhf_workspace_bytes(h) -> int:
    return int(lib().ddhf_workspace_bytes(h))


def ddhf_window(h, d_events_ptr: int, n: int, t0_us: int, window_us: int, d_workspace_ptr: int,
                out: DdhfOutputs, stream_ptr: int = 0) -> None:
    rc = lib().ddhf_window(h, d_events_ptr, n, t0_us, window_us, d_workspace_ptr, C.byref(out),
                           stream_ptr)
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(h) or b"").decode())


def ddhf_window_packed(h, d_events_ptr: int, n: int, t_base_us: int, t0_us: int, window_us: int, d_workspace_ptr: int,
                       out: DdhfOutputs, stream_ptr: int = 0) -> None:
    rc = lib().ddhf_window_packed(h, d_events_ptr, n, t_base_us, t0_us, window_us, d_workspace_ptr, C.byref(out),
                                  stream_ptr)
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(h) or b"").decode())


def ddhf_host_submit_packed(h, h_events_ptr: int, n: int, t_base_us: int, t0_us: int, window_us: int,
                            out: "DdhfHostOutputs", stream_ptr: int = 0) -> None:
    rc = lib().ddhf_host_submit_packed(h, h_events_ptr, n, t_base_us, t0_us, window_us, C.byref(out), stream_ptr)
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(h) or b"").decode())


def ddhf_window_slide(h, d_new_events_ptr: int, n_new: int, t0_us: int, window_us: int, d_workspace_ptr: int,
                      out: DdhfOutputs, stream_ptr: int = 0) -> None:
    rc = lib().ddhf_window_slide(h, d_new_events_ptr, n_new, t0_us, window_us, d_workspace_ptr, C.byref(out),
                                 stream_ptr)
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(h) or b"").decode())


def ddhf_slide_reset(h) -> None:
    lib().ddhf_slide_reset(h)


def ddhf_window_host(h, h_events_ptr: int, n: int, t0_us: int, window_us: int,
                     out: DdhfHostOutputs, stream_ptr: int = 0) -> None:
    rc = lib().ddhf_window_host(h, h_events_ptr, n, t0_us, window_us, C.byref(out), stream_ptr)
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(h) or b"").decode())


def ddhf_host_submit(h, h_events_ptr: int, n: int, t0_us: int, window_us: int,
                     out: DdhfHostOutputs, stream_ptr: int = 0) -> None:
    rc = lib().ddhf_host_submit(h, h_events_ptr, n, t0_us, window_us, C.byref(out), stream_ptr)
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(h) or b"").decode())


def ddhf_host_wait(h) -> None:
    rc = lib().ddhf_host_wait(h)
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(h) or b"").decode())


def ddhf_stage_ms(h) -> list[float]:
    ms = (C.c_float * 5)()
    rc = lib().ddhf_stage_ms(h, ms)
    if rc != DDHF_OK:
        raise DdhfError(rc, (lib().ddhf_last_error(h) or b"").decode())
    return [float(x) for x in ms]


NOALLOC_MAX_PIXELS, NOALLOC_MAX_BOXES = 921600, 4096


def ddhf_boxes_noalloc_setup() -> None:
    rc = lib().ddhf_boxes_noalloc_setup()
    if rc != DDHF_OK:
        raise DdhfError(rc, lib().ddhf_boxes_noalloc_error().decode())


def ddhf_boxes_noalloc(mask_ptr: int, width: int, height: int, a_min: int, merge_alpha: float, max_boxes: int,
                       labels_ptr: int, boxes_ptr: int, merged_ptr: int, counters_ptr: int, stream_ptr: int = 0) -> None:
    """ddhf.h: CCL + boxes (+ eq. 12) on a device mask with the library's static scratch; device pointers as ints."""
    rc = lib().ddhf_boxes_noalloc(mask_ptr, width, height, a_min, merge_alpha, max_boxes, labels_ptr, boxes_ptr,
                                  merged_ptr or None, counters_ptr, stream_ptr or None)
    if rc != DDHF_OK:
        raise DdhfError(rc, lib().ddhf_boxes_noalloc_error().decode())


def ddhf_launches_per_window(h) -> int:
    return int(lib().ddhf_launches_per_window(h))


def ddhf_fma_peak_probe(ms_target: float = 20.0, stream_ptr: int = 0) -> tuple[float, float]:
    out = (C.c_float * 2)()
    rc = lib().ddhf_fma_peak_probe(ms_target, out, stream_ptr)
    if rc != DDHF_OK:
        raise DdhfError(rc, "fma probe failed")
    return float(out[0]), float(out[1])


def ddhf_destroy(h) -> None:
    lib().ddhf_destroy(h)


def ddhf_version() -> str:
    return lib().ddhf_version().decode()


# ----------------------------------------------------------------------------------------
# convenience: a detector that owns torch buffers (allocation only -- no arithmetic)
# ----------------------------------------------------------------------------------------
class Detector:
    """Owns the handle, the workspace and the output tensors for one configuration."""

    def __init__(self, params: dict[str, Any], *, max_events: int, max_active: int | None = None,
                 max_boxes: int = 4096, max_scored: int = 0, score_all: bool = False, timing: bool = False,
                 want_power: bool = False, want_labels: bool = True, want_debug: bool = False,
                 nufft: bool = False, nufft_min: int = 0, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("DDHF needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        flags = (DDHF_FLAG_SCORE_ALL if score_all else 0) | (DDHF_FLAG_TIMING if timing else 0)
        if nufft:       # long rows by a non-uniform FFT (ddhf.h: DDHF_FLAG_NUFFT; bits 16-31: minimum row length)
            if not 0 <= nufft_min < 65536:
                raise ValueError("nufft_min must be in [0, 65535]")
            flags |= DDHF_FLAG_NUFFT | (int(nufft_min) << 16)
        self.params = dict(params)
        self.cfg = make_config(params, max_events=max_events, max_active=max_active,
                               max_boxes=max_boxes, max_scored=max_scored, flags=flags)
        self.h = ddhf_create(self.cfg)
        c = self.cfg
        self.np_ = c.width * c.height
        dev = self.device
        self.workspace = torch.empty(ddhf_workspace_bytes(self.h), dtype=torch.uint8, device=dev)
        z = lambda n, dt: torch.zeros(n, dtype=dt, device=dev)   # noqa: E731
        self.row_ptr = z(self.np_ + 1, torch.int32)
        self.csr_ev = z(max(c.max_events, 1), torch.int32)        # uint32 payload, viewed on the host
        self.active_idx = z(c.max_active, torch.int32)
        self.power = z(c.max_active * c.n_freq, torch.float32) if want_power else None
        self.sf = z(self.np_, torch.float32)
        self.score = z(self.np_, torch.float32)
        self.f0_idx = z(self.np_, torch.int32)
        self.mask = z(self.np_, torch.uint8)
        self.labels = z(self.np_, torch.int32) if want_labels else None
        self.boxes = z(c.max_boxes * 6, torch.int32)
        self.counters = z(N_COUNTERS, torch.int32)
        self.merged_boxes = z(c.max_boxes * 6, torch.int32) if c.merge_alpha > 0 else None
        self.comb_debug = z(c.max_active * c.n_f0 * 3, torch.float32) if want_debug else None
        o = DdhfOutputs()
        for name in ("row_ptr", "csr_ev", "active_idx", "power", "sf", "score", "f0_idx", "mask",
                     "labels", "boxes", "counters", "merged_boxes", "comb_debug"):
            t = getattr(self, name)
            setattr(o, name, None if t is None else t.data_ptr())
        self.out = o

    def upload(self, events: np.ndarray):
        """Host -> device copy of a 16-byte event array; returns a uint8 CUDA tensor."""
        torch = self.torch
        raw = np.ascontiguousarray(events).view(np.uint8)
        return torch.from_numpy(raw.copy()).to(self.device)

    def window(self, d_events, n: int, t0_us: int, window_us: int, *, offset_events: int = 0,
               stream=None) -> None:
        """Enqueue one window (asynchronous).  ``d_events``: uint8 CUDA tensor of event records."""
        torch = self.torch
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        ptr = d_events.data_ptr() + 16 * offset_events if n > 0 else 0
        ddhf_window(self.h, ptr, n, t0_us, window_us, self.workspace.data_ptr(), self.out,
                    st.cuda_stream)

    def window_packed(self, d_events8, n: int, t_base_us: int, t0_us: int, window_us: int, *, offset_events: int = 0,
                      stream=None) -> None:
        """ddhf_window on 8-byte events (``workloads.pack_events``): uint8 CUDA tensor of ddhf_event8 records."""
        torch = self.torch
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        ptr = d_events8.data_ptr() + 8 * offset_events if n > 0 else 0
        ddhf_window_packed(self.h, ptr, n, t_base_us, t0_us, window_us, self.workspace.data_ptr(), self.out,
                           st.cuda_stream)

    def slide(self, d_events, n_new: int, t0_us: int, window_us: int, *, offset_events: int = 0,
              stream=None) -> None:
        """Advance the sliding window kept in the workspace (ddhf_window_slide): ``n_new`` events starting
        at record ``offset_events`` of ``d_events`` are the events that follow those of the previous call."""
        torch = self.torch
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        ptr = d_events.data_ptr() + 16 * offset_events if n_new > 0 else 0
        ddhf_window_slide(self.h, ptr, n_new, t0_us, window_us, self.workspace.data_ptr(), self.out,
                          st.cuda_stream)

    def stage_ms(self) -> list[float]:
        return ddhf_stage_ms(self.h)

    def results(self) -> dict[str, Any]:
        """Synchronise and copy the outputs to numpy (device -> host)."""
        torch = self.torch
        torch.cuda.synchronize(self.device)
        c = self.cfg
        cnt = self.counters.cpu().numpy()
        n_in, n_act = int(cnt[CNT_N_IN]), min(int(cnt[CNT_N_ACTIVE]), c.max_active)
        n_box = int(cnt[CNT_N_BOXES])
        H, W = c.height, c.width
        res = dict(
            counters=cnt, n_in=n_in, n_dropped=int(cnt[CNT_N_DROPPED]),
            n_active=int(cnt[CNT_N_ACTIVE]), n_boxes=n_box, n_boxes_total=int(cnt[CNT_N_BOXES_TOTAL]),
            n_scored=int(cnt[CNT_N_SCORED]), overflow=int(cnt[CNT_OVERFLOW]),
            row_ptr=self.row_ptr.cpu().numpy(),
            csr_ev=self.csr_ev[:n_in].cpu().numpy().view(np.uint32),
            active_idx=self.active_idx[:n_act].cpu().numpy(),
            sf=self.sf.cpu().numpy().reshape(H, W), score=self.score.cpu().numpy().reshape(H, W),
            f0_idx=self.f0_idx.cpu().numpy().reshape(H, W),
            mask=self.mask.cpu().numpy().reshape(H, W),
            boxes=self.boxes[: n_box * 6].cpu().numpy().view(BOX_DTYPE).reshape(-1),
        )
        if self.merged_boxes is not None:
            n_m = int(cnt[CNT_N_MERGED])
            res["merged_boxes"] = self.merged_boxes[: n_m * 6].cpu().numpy().view(BOX_DTYPE).reshape(-1)
        if self.labels is not None:
            res["labels"] = self.labels.cpu().numpy().reshape(H, W)
        if self.power is not None:
            res["power"] = self.power[: n_act * c.n_freq].cpu().numpy().reshape(n_act, c.n_freq)
        if self.comb_debug is not None:
            res["comb_debug"] = self.comb_debug[: n_act * c.n_f0 * 3].cpu().numpy().reshape(n_act, c.n_f0, 3)
        return res

    def close(self) -> None:
        if self.h is not None:
            self.torch.cuda.synchronize(self.device)
            ddhf_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
