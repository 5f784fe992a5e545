"""Pins for the oracle's NDFT power (oracle/ddhf_oracle.c: orc_ndft_power, eq. 6).

None of these re-type the oracle's sum: they compare it with numpy's FFT on inputs where
the NDFT *is* a DFT, with closed forms, and with invariants the mathematics fixes.
"""
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_uniform_samples_reproduce_fft(oracle):
    # M events at t_k = k*T/M, f_j = j/T  ->  P = |fft(w)|^2  (north_star pin 1)
    rng = np.random.default_rng(1)
    M, T_us = 64, 64_000
    t = np.arange(M) * (T_us // M)
    w = rng.choice([-1.0, 1.0], size=M)
    P = oracle.ndft_power(t, w, 0.0, 1e6 / T_us, M)
    ref = np.abs(np.fft.fft(w)) ** 2
    assert np.max(np.abs(P - ref)) < 1e-9


def test_nonuniform_integer_timestamps_match_sparse_fft(oracle):
    # distinct integer-us timestamps < N, f_j = j * 1e6 / N Hz -> |fft(sparse sequence)|^2
    rng = np.random.default_rng(2)
    N = 4096
    t = np.sort(rng.choice(N, size=50, replace=False))
    w = rng.choice([-1.0, 1.0], size=50)
    seq = np.zeros(N)
    seq[t] = w
    ref = np.abs(np.fft.fft(seq)) ** 2
    P = oracle.ndft_power(t, w, 0.0, 1e6 / N, N)
    assert np.max(np.abs(P - ref)) < 1e-8
    # Parseval over the full DFT grid: mean_j P_j = sum w^2
    assert abs(P.mean() - 50.0) < 1e-9
    # a sub-grid with an offset start (f_min != 0) picks the same bins
    P2 = oracle.ndft_power(t, w, 100 * 1e6 / N, 2 * 1e6 / N, 500)
    assert np.max(np.abs(P2 - ref[100:1100:2])) < 1e-8


def test_unequal_weights_and_repeated_times(oracle):
    # general real weights (catches a dropped or squared weight); repeated timestamps add
    rng = np.random.default_rng(3)
    N = 1024
    t = rng.integers(0, N, size=200)
    w = rng.normal(size=200)
    seq = np.zeros(N)
    np.add.at(seq, t, w)
    ref = np.abs(np.fft.fft(seq)) ** 2
    P = oracle.ndft_power(t, w, 0.0, 1e6 / N, N)
    assert np.max(np.abs(P - ref)) < 1e-8 * max(1.0, ref.max())


def test_single_event_is_flat_w_squared(oracle):
    for w in (1.0, -1.0):
        P = oracle.ndft_power([12345], [w], 0.0, 4.8828125, 1024)
        assert np.allclose(P, 1.0, atol=1e-12)


def test_periodic_train_closed_form_and_golden(oracle):
    f0, tau, N = 200.0, 0.28, 20
    T0 = 1e6 / f0                                  # 5000 us, integer
    t_on = (np.arange(N) * T0).astype(np.int64)
    t_off = t_on + int(tau * T0)                   # 1400 us, integer
    t = np.concatenate([t_on, t_off])
    w = np.concatenate([np.ones(N), -np.ones(N)])
    # bins exactly on the harmonics
    P = oracle.ndft_power(t, w, 0.0, f0, 6)
    gold = np.loadtxt(os.path.join(GOLD, "periodic_train.txt"))
    for m, val in gold:
        m = int(m)
        assert abs(P[m] - 4 * N * N * math.sin(math.pi * m * tau) ** 2) < 1e-8
        assert abs(P[m] - val) < 2e-3              # golden file is printed to 3 decimals
    assert P[0] < 1e-20                            # DC: ON and OFF counts balance
    # all frequencies, grid not commensurate with 1/(N T0): Dirichlet kernel times pair factor
    df, nf = 7.3, 400
    f = np.arange(nf) * df
    P = oracle.ndft_power(t, w, 0.0, df, nf)
    with np.errstate(divide="ignore", invalid="ignore"):
        dirich = (np.sin(np.pi * f * N * T0 * 1e-6) / np.sin(np.pi * f * T0 * 1e-6)) ** 2
    dirich[0] = N * N
    ref = dirich * 4 * np.sin(np.pi * f * tau * T0 * 1e-6) ** 2
    assert np.max(np.abs(P - ref)) < 1e-7
    # peaks sit at k*f0: the largest bin within +-f0/2 of each harmonic is the nearest bin
    for m in (1, 2, 5):
        lo, hi = int((m - 0.5) * f0 / df), int((m + 0.5) * f0 / df)
        assert abs((lo + np.argmax(P[lo:hi])) * df - m * f0) <= df


def test_invariances(oracle):
    rng = np.random.default_rng(4)
    t = np.sort(rng.integers(0, 100_000, size=37))
    w = rng.choice([-1.0, 1.0], size=37)
    args = (0.0, 2.44140625, 512)
    P = oracle.ndft_power(t, w, *args)
    assert np.allclose(oracle.ndft_power(t + 777, w, *args), P, rtol=0, atol=1e-8)      # time shift
    assert np.allclose(oracle.ndft_power(t, -w, *args), P, rtol=0, atol=1e-10)          # polarity flip
    perm = rng.permutation(37)
    assert np.allclose(oracle.ndft_power(t[perm], w[perm], *args), P, rtol=0, atol=1e-9)  # order
    assert abs(P[0] - w.sum() ** 2) < 1e-12                                             # DC bin
    assert P.max() <= 37 ** 2 + 1e-9                                                    # |X| <= sum |w|
    # exponent sign (reading R1): conjugate spectrum, same power -- negative times mirror it
    assert np.allclose(oracle.ndft_power(100_000 - t, w, *args), P, rtol=0, atol=1e-8)


def test_tiny_bruteforce_cmath(oracle):
    import cmath
    t = [3, 1000, 1001, 5000, 7777, 9999, 12000, 20000]
    w = [1, -1, -1, 1, 1, -1, 1, 1]
    fmin, df, nf = 50.0, 37.5, 16
    P = oracle.ndft_power(t, w, fmin, df, nf)
    for j in range(nf):
        X = sum(wk * cmath.exp(-2j * cmath.pi * (fmin + j * df) * tk * 1e-6) for tk, wk in zip(t, w))
        assert abs(P[j] - abs(X) ** 2) < 1e-10
