"""Randomised GPU parity: random sensor sizes, grids, comb parameters, event mixes (hot pixels,
out-of-range events, unsorted input) against the oracle, every stage.  DDHF_FUZZ_SEEDS=n runs
n seeds instead of the default dozen."""
import os

import numpy as np
import pytest

from paper_2603_08386_b200 import workloads as wl

import gpu_util as gu

pytestmark = pytest.mark.gpu

N_SEEDS = int(os.environ.get("DDHF_FUZZ_SEEDS", "12"))
#: largest share of the active pixels that may be ill-conditioned, by n_min (1, 2, >= 3)
# n_min 2: a pixel with exactly two events has exact spectral nulls (opposite polarities: the DC bin; equal ones: every
# bin with f dt = 1/2 mod 1), and such pixels can be most of the active ones (seed 16: 302 of 360 active pixels hold two
# events, 273 are ill-conditioned); n_min >= 3: up to 44 % measured over 80 seeds
ILL_CAP = {1: 1.0, 2: 1.0, 3: 0.5}


def _case(seed):
    rng = np.random.default_rng([2603, 8386, 777, seed])
    W, H = int(rng.integers(8, 200)), int(rng.integers(8, 160))
    T = int(rng.choice([5_000, 20_000, 100_000, 1_000_000]))
    n = int(rng.integers(0, 60_000))
    nf = int(rng.choice([8, 40, 64, 130, 256, 300, 512, 700, 1024, 1500, 2048]))
    f_hi = float(rng.choice([500.0, 2000.0, 5000.0]))
    fmin = float(rng.choice([0.0, 0.0, 37.5]))
    df = (f_hi - fmin) / nf
    klo = int(rng.integers(0, 3)) if fmin == 0 else 0
    d = int(rng.integers(0, 4)) if nf >= 64 else 0
    n_harm = int(rng.integers(1, 7)) if nf >= 64 else 1
    f0_min = max(fmin + (d + klo + 2) * df, 20.0)
    prm = dict(width=W, height=H, window_us=T, f_min_hz=fmin, df_hz=df, n_freq=nf, k_lo=klo,
               f0_min_hz=f0_min, f0_step_hz=float(rng.choice([0.5, 2.0, 7.0])) * df,
               n_f0=int(rng.integers(1, 100)), n_harm=n_harm, half_bw_bins=d,
               h_min=int(rng.integers(1, n_harm + 1)), n_min=int(rng.integers(1, 8)),
               a_min=int(rng.integers(1, 12)), tau_sf=float(rng.uniform(0.3, 0.95)),
               tau_comb=float(rng.uniform(1.5, 8.0)), sf_eps=1e-12,
               merge_alpha=float(rng.choice([0.0, 1.0, 19.05])))
    ev = wl.random_window(1000 + seed, W, H, n, T, hot_fraction=float(rng.choice([0.0, 0.3, 0.8])),
                          out_of_range=float(rng.choice([0.0, 0.05])), time_sorted=bool(rng.integers(0, 2)))
    return prm, ev, T, bool(rng.integers(0, 2))


@pytest.mark.parametrize("seed", range(N_SEEDS))
def test_random_configuration(oracle, seed):
    from paper_2603_08386_b200 import binding
    prm, ev, T, score_all = _case(seed)
    try:
        gpu = gu.run_gpu(prm, ev, 0, T, score_all=score_all)
    except binding.DdhfError as e:
        # a configuration the library refuses at create time (comb windows too wide for the band
        # sorter) is not a parity case; anything else is a failure
        assert "band sorter" in str(e), str(e)
        pytest.skip(str(e))
    orc = oracle.window(prm, ev, 0, T, score_all=score_all)
    gu.check_csr(gpu, orc)
    assert gu.power_error(gpu["power"], orc["power"], gu.active_counts(orc)) <= gu.POWER_TOL
    # ill-conditioned pixels (R30): these streams are unstructured, so one- and two-event
    # pixels (exact spectral nulls) are the rule when n_min <= 2; the cap is a stated fraction of the
    # active pixels, and the count is printed
    n_act = max(int(orc["n_active"]), 1)
    gu.check_maps(gpu, orc, prm, score_all=score_all, oracle_mod=oracle, orc_power=orc["power"],
                  allow_ill=True, max_ill=int(ILL_CAP[min(prm["n_min"], 3)] * n_act) + 2)
    print(f"seed {seed}: n_min {prm['n_min']}, {gu.last_counts}")
    gu.check_boxes_against_oracle_ccl(gpu, oracle, prm["a_min"])


@pytest.mark.parametrize("seed", range(max(N_SEEDS // 2, 4)))
def test_random_bucketing_at_scale(oracle, seed):
    """CSR only, larger inputs: sensors up to 4 Mi pixels (digit widths from 6+6 to 11+11 bits), up to
    3 M events, several partition tiles with a ragged tail, skewed pixels, bad events, any order."""
    rng = np.random.default_rng([2603, 8386, 778, seed])
    W = int(rng.choice([64, 300, 640, 1280, 2048]))
    H = int(rng.choice([64, 200, 480, 720, 2048]))
    n = int(rng.choice([1, 8191, 8192, 8193, 100_000, 1_000_003, 3_000_000]))
    T = int(rng.choice([1000, 100_000, (1 << 31) - 1]))
    ev = wl.random_window(2000 + seed, W, H, n, T, hot_fraction=float(rng.choice([0.0, 0.5, 0.95])),
                          out_of_range=float(rng.choice([0.0, 0.1])), time_sorted=bool(rng.integers(0, 2)))
    t0 = int(rng.choice([0, 0, -12345]))
    ev["t"] += t0
    prm = dict(wl.preset(1), width=W, height=H, n_min=int(rng.integers(1, 5)))
    gpu = gu.run_gpu(prm, ev, t0, T, want_power=False, max_active=16)
    row_ptr, csr, dropped = oracle.bucket(ev, W, H, t0, T)
    assert gpu["n_dropped"] == dropped and gpu["n_in"] == len(csr)
    assert np.array_equal(gpu["row_ptr"], row_ptr), "row_ptr differs"
    assert np.array_equal(gpu["csr_ev"], csr), "csr_ev differs"
    cnt = np.diff(row_ptr)
    assert gpu["n_active"] == int((cnt >= prm["n_min"]).sum())
    assert np.array_equal(gpu["active_idx"], np.flatnonzero(cnt >= prm["n_min"])[:16])


def test_refused_configurations_are_rare():
    """`test_random_configuration` skips a draw that ddhf_create refuses (harmonic windows wider than the
    band sorter).  Those skips are counted here and capped: at most 10 % of the seeds."""
    from paper_2603_08386_b200 import binding
    refused = []
    for seed in range(N_SEEDS):
        prm, ev, T, score_all = _case(seed)
        try:
            binding.Detector(prm, max_events=16, want_power=False).close()
        except binding.DdhfError as e:
            assert "band sorter" in str(e), str(e)
            refused.append(seed)
    print(f"refused seeds (band sorter): {refused} of {N_SEEDS}")
    assert len(refused) <= max(1, N_SEEDS // 10)
