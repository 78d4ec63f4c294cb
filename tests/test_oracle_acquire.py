"""Pins of the oracle's initial range determination (reading R24).

What fixes it: a tone on an exact FFT bin (closed form: frequency exact, Hann-windowed amplitude A M/4), the known
accuracy of the log-parabolic refinement on a Hann window between bins, a direct DFT written as a matrix product
(independent of numpy.fft), a linear chirp (central difference = the chirp rate), and the one requirement the paper
states for the ranges: they "must cover the true value of parameters".
"""
import numpy as np
import pytest

import oracle
from paper_1906_10598_b200 import workloads as W


def test_tone_on_an_exact_bin():
    M, fs = 1024, 1024.0
    m = np.arange(M)
    for k, A, ph in ((37, 1.3, 0.4), (200, 0.5, -2.0), (1, 1.0, 0.0), (M // 2 - 1, 2.0, 1.0)):
        x = A * np.cos(2 * np.pi * k * m / M + ph)
        f, a, kp = oracle.piece_estimate(x, fs)
        assert kp == k
        if 1 < k < M // 2 - 1:                      # at the edge bins the mirror image overlaps the neighbours
            assert abs(f - k * fs / M) < 1e-9
            assert abs(a - A) < 1e-9 * A


def test_between_bins_accuracy_of_the_refinement():
    """Log-parabolic interpolation on a Hann window: frequency error < 0.02 bin, amplitude error < 1 %."""
    M, fs = 2048, 8000.0
    m = np.arange(M)
    worst_f = worst_a = 0.0
    for frac in np.linspace(-0.5, 0.5, 21):
        k0 = 300 + frac
        x = 0.8 * np.cos(2 * np.pi * k0 * m / M + 0.3)
        f, a, _ = oracle.piece_estimate(x, fs)
        worst_f = max(worst_f, abs(f * M / fs - k0))
        worst_a = max(worst_a, abs(a / 0.8 - 1))
    assert worst_f < 0.02 and worst_a < 0.01


def test_against_a_direct_dft():
    rng = np.random.default_rng(0)
    M, fs = 128, 128.0
    m = np.arange(M)
    x = np.cos(2 * np.pi * 20.3 * m / M + 1.0) + 0.1 * rng.standard_normal(M)
    w = 0.5 - 0.5 * np.cos(2 * np.pi * m / M)
    k = np.arange(M // 2 + 1)
    Xd = np.exp(-2j * np.pi * np.outer(k, m) / M) @ (x * w)
    P = np.abs(Xd) ** 2
    kp = 1 + int(np.argmax(P[1:M // 2]))
    lm, l0, lp = np.log(P[kp - 1]), np.log(P[kp]), np.log(P[kp + 1])
    delta = 0.5 * (lm - lp) / (lm - 2 * l0 + lp)
    f, a, kk = oracle.piece_estimate(x, fs)
    assert kk == kp == 20
    assert abs(f - (kp + delta) * fs / M) < 1e-10
    assert abs(a - 4 * np.sqrt(P[kp]) / M / (np.sinc(delta) / (1 - delta**2))) < 1e-10


def test_chirp_gives_fdot_by_central_difference():
    N, fs, M, S = 16000, 16000.0, 2048, 6000
    t = -0.5 + np.arange(N) / fs
    f0, fdot = 2000.3, 37.0
    x = 1.1 * np.cos(0.7 + 2 * np.pi * (f0 * t + fdot * t * t / 2))[None, :]
    r = oracle.acquire(x, fs, 5, M, S)
    a, fm, fc, fp, fd, *_ = r["est"][0]
    res = fs / M
    assert abs(fc - f0) < 0.05 * res
    assert abs(fm - (f0 - fdot * S / fs)) < 0.05 * res and abs(fp - (f0 + fdot * S / fs)) < 0.05 * res
    assert abs(fd - fdot) < 0.1 * res / (S / fs)
    assert abs(a - 1.1) < 0.02
    # ranges: items 1-6 of PAPER.md:181-187
    lo, hi = r["lo"][0], r["hi"][0]
    assert np.allclose([lo[0], hi[0]], [0.9 * a, 1.1 * a])
    assert np.allclose([lo[1], hi[1]], [-0.2 * a / 1.0, 0.2 * a / 1.0])
    assert np.allclose([lo[2], hi[2]], [-np.pi, np.pi])
    assert np.allclose([lo[3], hi[3]], [0.9 * fc, 1.1 * fc])
    assert np.allclose([lo[4], hi[4]], [fd - res / (S / fs), fd + res / (S / fs)])
    r6 = oracle.acquire(x, fs, 6, M, S, f_rel=0.0, f_bins=2.0)
    assert np.allclose([r6["lo"][0, 5], r6["hi"][0, 5]], [-150 / np.pi, 150 / np.pi])   # c3 in [-50, 50], c3 = (pi/3) fddot
    assert np.allclose([r6["lo"][0, 3], r6["hi"][0, 3]], [fc - 2 * res, fc + 2 * res])


@pytest.mark.parametrize("name", ["config0", "config1", "config2"])
def test_ranges_cover_the_truth(name):
    """the ranges "must cover the true value of parameters"."""
    if name == "config0":
        wl, M = W.config0(cases=range(16)), 256
    elif name == "config1":
        wl, M = W.config1(blocks=[0, 20, 40, 59]), 2048
    else:
        wl, M = W.config2(blocks=[0, 900, 1800, 2700, 3599]), 4096
    S = (wl.N - M) // 2
    r = oracle.acquire(wl.x, wl.fs, wl.D, M, S, f_rel=0.0, f_bins=1.0, fdot_bins=2.0, a_rel=0.2)
    th = wl.truth
    for j in (0, 1, 3, 4):
        assert np.all(r["lo"][:, j] <= th[:, j]) and np.all(th[:, j] <= r["hi"][:, j]), (name, j)
    # and with the paper's own +-10 % of c1
    r = oracle.acquire(wl.x, wl.fs, wl.D, M, S)
    assert np.all(r["lo"][:, 3] <= th[:, 3]) and np.all(th[:, 3] <= r["hi"][:, 3])


def test_invalid_arguments():
    x = np.zeros((1, 1000), dtype=np.float32)
    for M, S in ((100, 10), (512, 300), (4, 10)):
        with pytest.raises(ValueError):
            oracle.acquire(x, 1000.0, 5, M, S)
