"""Pins for the oracle's bucketing (a0-a3), CCL/boxes (a8) and the whole window.

Bucketing is pinned to numpy's stable argsort / bincount / cumsum, CCL to
scipy.ndimage.label with the 8-connected structure; the whole-window call is pinned by
recomposing it from the separately pinned stage functions and by the generator's ground
truth on config 1.
"""
import numpy as np
import pytest
from scipy import ndimage

from paper_2603_08386_b200 import workloads as wl


def test_bucket_matches_numpy_stable_sort(oracle):
    W, H, T = 37, 23, 10_000
    ev = wl.random_window(1, W, H, 5000, T, hot_fraction=0.3, out_of_range=0.1, time_sorted=False)
    t0 = 0
    row_ptr, csr, dropped = oracle.bucket(ev, W, H, t0, T)
    ok = (ev["t"] >= t0) & (ev["t"] < t0 + T) & (ev["x"] < W) & (ev["y"] < H)
    assert dropped == int((~ok).sum()) and dropped > 100
    kept = ev[ok]
    key = kept["y"].astype(np.int64) * W + kept["x"]
    order = np.argsort(key, kind="stable")
    want_val = ((kept["t"][order] - t0).astype(np.uint32) << 1) | (kept["p"][order] > 0)
    want_ptr = np.concatenate([[0], np.cumsum(np.bincount(key, minlength=W * H))])
    assert np.array_equal(row_ptr, want_ptr)
    assert np.array_equal(csr, want_val.astype(np.uint32))


def test_bucket_window_edges_and_t0(oracle):
    ev = np.zeros(4, dtype=wl.EVENT_DTYPE)
    ev["t"] = [999, 1000, 1999, 2000]
    ev["p"] = [1, -1, 1, 1]
    row_ptr, csr, dropped = oracle.bucket(ev, 2, 2, 1000, 1000)   # [t0, t0 + window)
    assert dropped == 2 and list(csr) == [(0 << 1) | 0, (999 << 1) | 1]
    # p = 0 counts as negative (p > 0 -> +1 else -1, reading R21)
    ev["p"][2] = 0
    assert oracle.bucket(ev, 2, 2, 1000, 1000)[1][1] == (999 << 1)


def test_bucket_empty(oracle):
    ev = np.zeros(0, dtype=wl.EVENT_DTYPE)
    row_ptr, csr, dropped = oracle.bucket(ev, 8, 8, 0, 100)
    assert row_ptr.sum() == 0 and len(csr) == 0 and dropped == 0


def _scipy_boxes(mask, a_min):
    lab, n = ndimage.label(mask, structure=np.ones((3, 3), int))
    out = []
    for i, sl in enumerate(ndimage.find_objects(lab), start=1):
        ys, xs = sl
        comp = np.flatnonzero((lab == i).ravel())
        area = (xs.stop - xs.start) * (ys.stop - ys.start)
        if area >= a_min:
            out.append((xs.start, ys.start, xs.stop - 1, ys.stop - 1, len(comp), int(comp.min())))
    return sorted(out, key=lambda b: b[5]), lab


@pytest.mark.parametrize("density", [0.05, 0.3, 0.6])
def test_ccl_matches_scipy(oracle, density):
    rng = np.random.default_rng(int(density * 100))
    mask = rng.random((61, 83)) < density
    for a_min in (1, 9):
        labels, boxes, tot = oracle.ccl_boxes(mask, a_min)
        want, lab = _scipy_boxes(mask, a_min)
        got = [tuple(int(b[k]) for k in ("x0", "y0", "x1", "y1", "n_pix", "label")) for b in boxes]
        assert got == want and tot == len(want)
    # same partition: oracle label = min linear index of scipy's component
    flat = lab.ravel()
    mins = ndimage.minimum(np.arange(flat.size), flat, index=np.arange(1, flat.max() + 1))
    want_lab = np.where(flat > 0, np.asarray(mins, dtype=np.int64)[np.maximum(flat, 1) - 1], -1)
    assert np.array_equal(labels.ravel(), want_lab)


def test_ccl_diagonal_touch_joins(oracle):
    m = np.zeros((4, 4), bool)
    m[0, 0] = m[1, 1] = m[2, 2] = True      # diagonal chain: one component under 8-connectivity
    m[0, 3] = True                          # isolated
    labels, boxes, _ = oracle.ccl_boxes(m, 1)
    assert len(boxes) == 2
    assert tuple(boxes[0])[:5] == (0, 0, 2, 2, 3) and boxes[0]["label"] == 0
    assert tuple(boxes[1])[:5] == (3, 0, 3, 0, 1) and boxes[1]["label"] == 3
    # bounding-box area, not pixel count (reading R17): the chain has 3 px but area 9
    assert len(oracle.ccl_boxes(m, 9)[1]) == 1
    assert len(oracle.ccl_boxes(m, 10)[1]) == 0


def test_ccl_empty_and_full(oracle):
    assert len(oracle.ccl_boxes(np.zeros((5, 7), bool), 1)[1]) == 0
    labels, boxes, _ = oracle.ccl_boxes(np.ones((5, 7), bool), 1)
    assert len(boxes) == 1 and tuple(boxes[0]) == (0, 0, 6, 4, 35, 0) and (labels == 0).all()


def test_box_cap(oracle):
    m = np.zeros((9, 9), bool)
    m[::2, ::2] = True
    labels, boxes, tot = oracle.ccl_boxes(m, 1, max_boxes=7)
    assert len(boxes) == 7 and tot == 25 and list(boxes["label"]) == sorted(boxes["label"])


@pytest.mark.parametrize("score_all", [False, True])
def test_window_is_the_composition_of_the_stages(oracle, score_all):
    w = wl.make(1)
    prm = dict(w.params, n_min=3)
    out = oracle.window(prm, w.events, 0, w.window_us, score_all=score_all)
    row_ptr, csr, dropped = oracle.bucket(w.events, w.width, w.height, 0, w.window_us)
    assert np.array_equal(out["row_ptr"], row_ptr) and np.array_equal(out["csr_ev"], csr)
    assert out["n_dropped"] == dropped and out["n_in"] == len(csr)
    cnt = np.diff(row_ptr)
    act = np.flatnonzero(cnt >= 3)
    assert np.array_equal(out["active_idx"], act) and out["n_active"] == len(act)
    mask = np.zeros(w.width * w.height, np.uint8)
    for r, p in enumerate(act):
        seg = csr[row_ptr[p]:row_ptr[p + 1]]
        P = oracle.ndft_power(seg >> 1, np.where(seg & 1, 1.0, -1.0), prm["f_min_hz"],
                              prm["df_hz"], prm["n_freq"])
        assert np.array_equal(out["power"][r], P)
        sf = oracle.spectral_flatness(P, prm["k_lo"], prm["sf_eps"])
        y, x = divmod(int(p), w.width)
        assert out["sf"][y, x] == sf
        if score_all or sf <= prm["tau_sf"]:
            s, fi, *_ = oracle.comb_score(P, prm)
            assert out["score"][y, x] == s and out["f0_idx"][y, x] == fi
            mask[p] = sf <= prm["tau_sf"] and fi >= 0 and s >= prm["tau_comb"]
        else:
            assert out["score"][y, x] == 0.0 and out["f0_idx"][y, x] == -1
    assert np.array_equal(out["mask"].ravel(), mask)
    inactive = np.ones(w.width * w.height, bool)
    inactive[act] = False
    assert np.isnan(out["sf"].ravel()[inactive]).all() and (out["f0_idx"].ravel()[inactive] == -1).all()
    labels, boxes, _ = oracle.ccl_boxes(mask.reshape(w.height, w.width), prm["a_min"])
    assert np.array_equal(out["labels"], labels) and np.array_equal(out["boxes"], boxes)


def test_config1_ground_truth(oracle):
    """End-to-end sanity (not parity): the 8x8 rotor patch is found, f0 within one step."""
    w = wl.make(1)
    out = oracle.window(w.params, w.events, 0, w.window_us)
    truth = w.truth["mask"]
    hit = out["mask"].astype(bool) & truth
    assert hit.sum() >= 0.8 * truth.sum()
    assert (out["mask"].astype(bool) & ~truth).sum() <= 2
    f0 = w.params["f0_min_hz"] + out["f0_idx"][hit] * w.params["f0_step_hz"]
    assert np.median(np.abs(f0 - 200.0)) <= w.params["f0_step_hz"]
    assert len(out["boxes"]) == 1
    b = out["boxes"][0]
    assert 38 <= b["x0"] <= 42 and 45 <= b["x1"] <= 49 and 22 <= b["y0"] <= 26 and 29 <= b["y1"] <= 33


# ---- box merge (eq. 12) --------------------------------------------------------------------
def _boxes(rows):
    import ddhf_oracle
    b = np.zeros(len(rows), dtype=ddhf_oracle.ORC_BOX)
    for i, (x0, y0, x1, y1) in enumerate(rows):
        b[i] = (x0, y0, x1, y1, (x1 - x0 + 1) * (y1 - y0 + 1), y0 * 10000 + x0)
    return b


def test_merge_far_near_and_chain(oracle):
    # two 10x10 boxes 100 px apart: dist 100 >= alpha*10 for alpha 5 -> separate; alpha 11 -> merged
    b = _boxes([(0, 0, 9, 9), (100, 0, 109, 9)])
    assert len(oracle.merge_boxes(b, 5.0)) == 2
    m = oracle.merge_boxes(b, 11.0)
    assert len(m) == 1 and (m[0]["x0"], m[0]["y0"], m[0]["x1"], m[0]["y1"]) == (0, 0, 109, 9)
    assert m[0]["n_pix"] == 200 and m[0]["label"] == b[0]["label"]
    # exactly on the threshold is NOT merged (strict <): dist 100, alpha*max = 10*10
    assert len(oracle.merge_boxes(b, 10.0)) == 2
    # chain A~B, B~C but A !~ C: transitive -> one box (R28)
    c = _boxes([(0, 0, 9, 9), (60, 0, 69, 9), (120, 0, 129, 9)])
    assert len(oracle.merge_boxes(c, 6.5)) == 1 and len(oracle.merge_boxes(c, 5.9)) == 3
    # the larger box sets the scale: a 40-wide box reaches a small one that could not reach it alone
    d = _boxes([(0, 0, 39, 3), (100, 0, 101, 1)])
    assert len(oracle.merge_boxes(d, 2.5)) == 1            # centre distance 81 < 2.5 * 40
    assert len(oracle.merge_boxes(_boxes([(0, 0, 1, 1), (100, 0, 101, 1)]), 2.5)) == 2
    assert len(oracle.merge_boxes(_boxes([]), 3.0)) == 0


def test_merge_matches_connected_components_of_the_close_relation(oracle):
    """Independent construction: adjacency by eq. 12 in numpy, components by scipy.sparse.csgraph."""
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import connected_components
    rng = np.random.default_rng(12)
    for alpha in (0.8, 2.0, 4.0):
        rows = []
        for _ in range(60):
            x0, y0 = int(rng.integers(0, 600)), int(rng.integers(0, 400))
            rows.append((x0, y0, x0 + int(rng.integers(1, 30)), y0 + int(rng.integers(1, 30))))
        rows.sort(key=lambda r: r[1] * 10000 + r[0])
        b = _boxes(rows)
        cx, cy = (b["x0"] + b["x1"]) / 2.0, (b["y0"] + b["y1"]) / 2.0
        dim = np.maximum(b["x1"] - b["x0"] + 1, b["y1"] - b["y0"] + 1).astype(float)
        dist = np.hypot(cx[:, None] - cx[None, :], cy[:, None] - cy[None, :])
        adj = dist < alpha * np.maximum(dim[:, None], dim[None, :])
        n_comp, lab = connected_components(csr_matrix(adj), directed=False)
        m = oracle.merge_boxes(b, alpha)
        assert len(m) == n_comp
        for k in range(n_comp):
            members = b[lab == k]
            hit = m[m["label"] == members["label"].min()]
            assert len(hit) == 1
            assert hit[0]["x0"] == members["x0"].min() and hit[0]["x1"] == members["x1"].max()
            assert hit[0]["y0"] == members["y0"].min() and hit[0]["y1"] == members["y1"].max()
            assert hit[0]["n_pix"] == members["n_pix"].sum()
        assert np.all(np.diff(m["label"]) > 0)
