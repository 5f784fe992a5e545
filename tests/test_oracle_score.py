"""Pins for the oracle's spectral flatness (eq. 7) and median-normalised comb (eq. 8-11).

Hand-built spectra whose flatness, comb numerator, complement median and SNR are known in
closed form; each case is chosen so that one plausible slip (window edge off by one, mean
vs. median, union vs. sum of windows, upper vs. lower median, dropped harmonic, wrong
validity rule) changes the expected number.
"""
import math

import numpy as np
import pytest

BASE = dict(width=1, height=1, f_min_hz=0.0, df_hz=10.0, n_freq=201, f0_min_hz=100.0,
            f0_step_hz=10.0, n_f0=31, n_harm=5, half_bw_bins=2, h_min=4, n_min=1, a_min=1,
            tau_sf=1.0, tau_comb=0.0, sf_eps=1e-12, k_lo=1)


# ---------------------------------------------------------------- spectral flatness
def test_sf_flat_is_one_and_scale_invariant(oracle):
    for c in (1.0, 7.5, 1e-6):
        assert abs(oracle.spectral_flatness(np.full(300, c), 1, 1e-12) - 1.0) < 1e-12


def test_sf_single_spike_closed_form(oracle):
    n, A = 200, 50.0
    P = np.ones(n + 1)          # bin 0 is skipped by k_lo = 1
    P[0] = 1e9                  # must not matter
    P[17] = A
    want = A ** (1.0 / n) / ((n - 1 + A) / n)
    assert abs(oracle.spectral_flatness(P, 1, 1e-12) - want) < 1e-12
    # k_lo = 0 includes the DC bin
    P[0] = 1.0
    want0 = A ** (1.0 / (n + 1)) / ((n + A) / (n + 1))
    assert abs(oracle.spectral_flatness(P, 0, 1e-12) - want0) < 1e-12


def test_sf_floor_on_zero_power(oracle):
    P = np.ones(101)
    P[5] = 0.0                  # log(0) is floored at eps (reading R6)
    eps = 1e-12
    want = math.exp(math.log(eps) / 100) / ((99 + eps) / 100)
    assert abs(oracle.spectral_flatness(P, 1, eps) - want) < 1e-12


def test_sf_white_noise_expectation(oracle):
    # exponential powers (chi^2_2): E[SF] -> exp(-gamma) = 0.5615 (statistical sanity)
    rng = np.random.default_rng(5)
    vals = [oracle.spectral_flatness(rng.exponential(size=4096), 0, 1e-12) for _ in range(20)]
    assert abs(np.mean(vals) - math.exp(-0.5772156649)) < 0.01


# ---------------------------------------------------------------- comb
def comb_spectrum(f0, A=9.0, n_harm=5, df=10.0, nf=201):
    P = np.ones(nf)
    for m in range(1, n_harm + 1):
        k = int(math.floor(m * f0 / df + 0.5))
        if k < nf:
            P[k] = A
    return P


def test_comb_known_numerator_median_snr(oracle):
    P = comb_spectrum(200.0, A=9.0)
    s, fi, snr, num, med = oracle.comb_score(P, BASE)
    c200 = 10                                     # (200 - 100) / 10
    assert num[c200] == 9.0 and med[c200] == 1.0 and snr[c200] == 9.0
    assert fi == c200 and s == 9.0
    # candidate 100 Hz sees spikes only at even harmonics 2, 4 of its own comb: (1+9+1+9+1)/5
    assert abs(num[0] - 21.0 / 5) < 1e-12
    # candidate 400 Hz: its harmonics 1, 2 hit 400 and 800 (spikes), 3.. hit floor; 5*400 = 2000
    # -> window [198, 202] leaves the band, so M_valid = 4 and N = (9 + 9 + 1 + 1) / 4
    assert abs(num[30] - 20.0 / 4) < 1e-12


def test_comb_second_rotor_does_not_move_the_median(oracle):
    # two rotors on one pixel: the second comb raises the mean of the
    # complement but not its median
    P = comb_spectrum(200.0, A=9.0)
    for m in range(1, 6):
        P[int(round(m * 17.0))] = 30.0            # 170 Hz comb, 5 strong lines
    s, fi, snr, num, med = oracle.comb_score(P, BASE)
    assert med[10] == 1.0 and snr[10] == 9.0
    comp_mean = (P[1:].sum() - 5 * 9.0 - 20 * 1.0) / (200 - 25)
    assert comp_mean > 1.5                        # a mean-normalised SNR would have dropped


def test_comb_window_edges(oracle):
    d = BASE["half_bw_bins"]
    for off, inside in ((d, True), (-d, True), (d + 1, False), (-d - 1, False)):
        P = np.ones(201)
        P[20 + off] = 5.0                         # near harmonic 1 of 200 Hz (bin 20)
        _, _, snr, num, med = oracle.comb_score(P, BASE)
        want = (5.0 + 4.0) / 5 if inside else 1.0
        assert abs(num[10] - want) < 1e-12, (off, num[10])


def test_comb_validity_prefix_and_hmin(oracle):
    P = np.ones(201)
    prm = dict(BASE, f0_min_hz=100.0, f0_step_hz=10.0, n_f0=41, n_harm=5, h_min=4)
    _, _, snr, num, med = oracle.comb_score(P, prm)
    # f0 = 490 Hz: 4*490 = 1960 -> window [194,198] in band, 5*490 out  -> M_valid = 4, kept
    assert snr[39] == 1.0
    # f0 = 500 Hz: 4*500 = 2000 -> bin 200, window [198,202] out of band -> M_valid = 3 < h_min
    assert snr[40] == 0.0
    # flat spectrum everywhere valid -> SNR exactly 1, first candidate wins ties (R16)
    s, fi, *_ = oracle.comb_score(P, prm)
    assert s == 1.0 and fi == 0
    # lower band edge: with k_lo = 9 the first window of f0 = 100 Hz ([8,12]) is out -> skipped
    _, _, snr2, *_ = oracle.comb_score(P, dict(prm, k_lo=9))
    assert snr2[0] == 0.0 and snr2[1] == 1.0
    # nothing valid at all -> score 0, index -1
    s3, fi3, *_ = oracle.comb_score(P, dict(prm, h_min=6))
    assert s3 == 0.0 and fi3 == -1


def test_comb_lower_median_even_count_and_union(oracle):
    # values 1..200 on bins 1..200: complement of a candidate = those values minus its windows
    nf = 201
    P = np.zeros(nf)
    P[1:] = np.arange(1, nf, dtype=float)
    prm = dict(BASE, half_bw_bins=5, n_harm=5, h_min=4)      # f0 = 100: windows [5,15],[15,25],.. overlap at one bin
    _, _, snr, num, med = oracle.comb_score(P, prm)
    # f0 = 100 Hz: centres 10,20,30,40,50, windows [5,15]..[45,55] -> union = bins 5..55 (51 bins)
    comp = [v for v in range(1, 201) if not (5 <= v <= 55)]
    assert len(comp) == 149
    assert med[0] == sorted(comp)[(len(comp) - 1) // 2]
    assert num[0] == (15 + 25 + 35 + 45 + 55) / 5
    # f0 = 200 Hz: centres 20..100 step 20, windows disjoint -> 55 bins out, 145 left (odd)
    comp = [v for v in range(1, 201) if not any(abs(v - c) <= 5 for c in (20, 40, 60, 80, 100))]
    assert med[10] == sorted(comp)[(len(comp) - 1) // 2]
    # f0 = 390 Hz: M_valid = 5 (5*390 = 1950 -> [190,200] in band); 200 - 55 = 145 left
    # f0 = 400 Hz: 5*400 = 2000 -> out, M_valid = 4 -> 44 bins out -> 156 left (EVEN count)
    comp = [v for v in range(1, 201) if not any(abs(v - c) <= 5 for c in (40, 80, 120, 160))]
    assert len(comp) % 2 == 0
    assert med[30] == sorted(comp)[len(comp) // 2 - 1]       # lower of the two middle values (R10)


def test_comb_noninteger_harmonic_centres(oracle):
    # df = 4.8828125 Hz: centre bin = floor(m f0 / df + 0.5)  (reading R7)
    df = 5000.0 / 1024
    prm = dict(BASE, df_hz=df, n_freq=1024, f0_min_hz=100.0, f0_step_hz=5.0, n_f0=81, n_harm=6,
               half_bw_bins=0, h_min=4)
    f0 = 235.0
    P = np.ones(1024)
    ks = [int(math.floor(m * f0 / df + 0.5)) for m in range(1, 7)]
    for k in ks:
        P[k] = 4.0
    s, fi, snr, num, med = oracle.comb_score(P, prm)
    assert fi == 27 and num[27] == 4.0 and s == 4.0          # with d = 0 only exact centres count
    P2 = np.ones(1024)
    for k in ks:
        P2[k + 1] = 4.0
    assert oracle.comb_score(P2, prm)[3][27] == 1.0


def test_comb_median_floor(oracle):
    P = np.zeros(201)
    P[20] = 3.0
    _, _, snr, num, med = oracle.comb_score(P, BASE)
    assert med[10] == 0.0 and snr[10] == pytest.approx((3.0 / 5) / 1e-12)   # R11
