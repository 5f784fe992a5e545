"""ddhf_boxes_noalloc (include/ddhf.h): CCL + boxes + eq. 12 detections with the library's static scratch, against
the existing path (ddhf_window with a caller's workspace) on the same masks.  Integer work: bit-exact.  Collected
last on purpose (the suite runs with pytest -x).  Run with `pytest -m gpu` on a B200."""
import numpy as np
import pytest

from paper_2603_08386_b200 import workloads as wl

import gpu_util as gu

pytestmark = pytest.mark.gpu


def _existing_path(w, params):
    res = gu.run_gpu(params, w.events, w.t0_us, w.window_us, want_power=False)
    assert "merged_boxes" in res and "labels" in res
    return res


def _noalloc(binding, torch, ref, params, max_boxes=4096):
    """One call of the new entry point on the mask of `ref`; returns what it wrote."""
    dev = torch.device("cuda:0")
    H, W = ref["mask"].shape
    mask = torch.from_numpy(np.ascontiguousarray(ref["mask"])).to(dev)
    # outputs start as garbage: the call must not depend on their contents
    labels = torch.full((H * W,), 12345, dtype=torch.int32, device=dev)
    boxes = torch.full((max_boxes * 6,), -7, dtype=torch.int32, device=dev)
    merged = torch.full((max_boxes * 6,), -7, dtype=torch.int32, device=dev)
    counters = torch.full((binding.N_COUNTERS,), 99, dtype=torch.int32, device=dev)
    binding.ddhf_boxes_noalloc(mask.data_ptr(), W, H, int(params["a_min"]), float(np.float32(params["merge_alpha"])), max_boxes,
                               labels.data_ptr(), boxes.data_ptr(), merged.data_ptr(), counters.data_ptr(),
                               torch.cuda.current_stream(dev).cuda_stream)
    torch.cuda.synchronize(dev)
    cnt = counters.cpu().numpy()
    nb, nm = int(cnt[binding.CNT_N_BOXES]), int(cnt[binding.CNT_N_MERGED])
    return dict(counters=cnt, labels=labels.cpu().numpy().reshape(H, W),
                boxes=boxes[: nb * 6].cpu().numpy().view(binding.BOX_DTYPE).reshape(-1),
                merged_boxes=merged[: nm * 6].cpu().numpy().view(binding.BOX_DTYPE).reshape(-1))


def _same(binding, got, ref):
    for k in (binding.CNT_N_BOXES, binding.CNT_N_BOXES_TOTAL, binding.CNT_N_COMPONENTS, binding.CNT_N_MERGED):
        assert got["counters"][k] == ref["counters"][k], (k, got["counters"], ref["counters"])
    assert (got["counters"][binding.CNT_OVERFLOW] & 2) == (ref["counters"][binding.CNT_OVERFLOW] & 2)
    assert np.array_equal(got["labels"], ref["labels"])
    assert np.array_equal(got["boxes"], ref["boxes"])
    assert np.array_equal(got["merged_boxes"], ref["merged_boxes"])


def test_noalloc_boxes_match_the_workspace_path_on_calls_in_a_row():
    import torch
    from paper_2603_08386_b200 import binding
    binding.ddhf_boxes_noalloc_setup()
    wa = wl.make(4, scale=0.25)                  # 320 x 180, about a thousand mask pixels
    # Table 2's thresholds put noise pixels into the mask too: many components, many of them below A_min
    pa = dict(wa.params, tau_sf=0.89, tau_comb=1.5, a_min=4)
    wb = wl.make(1)                              # 64 x 64: another sensor size right after, on the same scratch
    wc = wl.make(4)                              # 1280 x 720: the largest sensor the static scratch holds
    ref_a, ref_b, ref_c = _existing_path(wa, pa), _existing_path(wb, wb.params), _existing_path(wc, wc.params)
    assert ref_a["counters"][binding.CNT_N_COMPONENTS] > 20 and len(ref_a["boxes"]) >= 2
    assert len(ref_b["boxes"]) >= 1
    assert ref_c["mask"].size == binding.NOALLOC_MAX_PIXELS and len(ref_c["boxes"]) >= 2

    def series():
        _same(binding, _noalloc(binding, torch, ref_a, pa), ref_a)
        # second call in a row: the array holds the leftovers of the first
        _same(binding, _noalloc(binding, torch, ref_b, wb.params), ref_b)
        _same(binding, _noalloc(binding, torch, ref_c, wc.params), ref_c)
        _same(binding, _noalloc(binding, torch, ref_a, pa), ref_a)
        got = _noalloc(binding, torch, ref_a, pa, max_boxes=1)   # boxes beyond max_boxes: counted, flagged, not written
        assert got["counters"][binding.CNT_OVERFLOW] & 2 and len(got["boxes"]) == 1
        assert got["counters"][binding.CNT_N_BOXES_TOTAL] == ref_a["counters"][binding.CNT_N_BOXES_TOTAL]
        assert np.array_equal(got["boxes"], ref_a["boxes"][:1])

    series()
    # nothing is allocated on the device by the calls: the second pass finds the test's own tensors in torch's pool
    free0 = torch.cuda.mem_get_info(0)[0]
    series()
    assert torch.cuda.mem_get_info(0)[0] >= free0 - (2 << 20)
    print(f"noalloc: {len(ref_a['boxes'])} boxes / {len(ref_a['merged_boxes'])} detections of "
          f"{ref_a['counters'][binding.CNT_N_COMPONENTS]} components (320x180), {len(ref_b['boxes'])} boxes (64x64), "
          f"{len(ref_c['boxes'])} boxes (1280x720): identical")


def test_noalloc_empty_mask_and_limits():
    import torch
    from paper_2603_08386_b200 import binding
    dev = torch.device("cuda:0")
    ref = dict(mask=np.zeros((48, 40), np.uint8))
    got = _noalloc(binding, torch, ref, dict(a_min=1, merge_alpha=19.05))
    assert (got["labels"] == -1).all() and len(got["boxes"]) == 0 and len(got["merged_boxes"]) == 0
    assert not got["counters"].any()
    z = torch.zeros(64, dtype=torch.int32, device=dev)
    for w, h, mb in ((1281, 720, 16), (1280, 721, 16), (64, 64, 4097), (64, 64, 0)):
        with pytest.raises(binding.DdhfError) as ei:
            binding.ddhf_boxes_noalloc(z.data_ptr(), w, h, 1, 0.0, mb, z.data_ptr(), z.data_ptr(), 0, z.data_ptr(), 0)
        assert ei.value.code == binding.DDHF_E_CAPACITY and "DDHF_NOALLOC_MAX" in str(ei.value)
    with pytest.raises(binding.DdhfError) as ei:
        binding.ddhf_boxes_noalloc(0, 64, 64, 1, 0.0, 16, z.data_ptr(), z.data_ptr(), 0, z.data_ptr(), 0)
    assert ei.value.code == binding.DDHF_E_INVAL
