"""Pins of the oracle's correlation objective (Eq. 5-6; reading R22).

    F_cor = 1 / (arctan(cor(s_i, s(c_k, t_i))) + pi/2),   s(t) = A cos(c0 + c1 t + c2 t^2 + c3 t^3)

What the paper fixes: F_cor "shall converge to 1/pi ~ 0.318" and the constant it subtracts for
display, 0.31830988618 (tests/golden/fcor_limit.txt).  What the mathematics fixes: closed forms
of the correlation sum on whole cycles of a tone, its symmetries, and that on a constant-amplitude signal its
maximiser is the least-squares phase.
"""
import os

import numpy as np
import pytest
from scipy.optimize import least_squares

import oracle
from paper_1906_10598_b200 import workloads as W


def test_limit_printed_by_the_paper(golden_dir):
    """the objective tends to 1/pi, printed as 0.31830988618."""
    with open(os.path.join(golden_dir, "fcor_limit.txt")) as fh:
        printed = [float(line.split()[0]) for line in fh if line.strip() and not line.startswith("#")]
    assert printed == [0.31830988618]
    for c in (1e9, 1e12, 1e15):
        assert abs(oracle.fcor_of_cor(c) - printed[0]) < 0.5e-11 + 1.1 / (np.pi**2 * c)
    # and it is approached from above: F_cor - 1/pi = 1/(pi^2 cor) to first order
    for c in (1e3, 1e5):
        assert abs((oracle.fcor_of_cor(c) - 1 / np.pi) * np.pi**2 * c - 1) < 2 / c + 1e-9


def test_eq5_special_values_and_monotonicity():
    assert oracle.fcor_of_cor(0.0) == 2 / np.pi                       # arctan 0 = 0
    assert abs(oracle.fcor_of_cor(1.0) - 1 / (np.pi / 4 + np.pi / 2)) < 1e-16
    assert abs(oracle.fcor_of_cor(-1.0) - 1 / (np.pi / 4)) < 1e-15
    c = np.linspace(-50, 5000, 2001)
    f = np.array([oracle.fcor_of_cor(v) for v in c])
    assert np.all(np.diff(f) < 0)                                     # strictly decreasing: min F_cor = max cor
    assert np.all(f > 1 / np.pi)


def test_closed_form_on_whole_cycles():
    """x = A cos(phi0 + 2 pi f t) over an integer number of cycles (N even, f = k fs/N, 0 < k < N/2):
    sum x * a0 cos(phi0 + 2 pi f t + d) = a0 A (N/2) cos d."""
    N, fs, k = 400, 400.0, 37
    t = -N / (2 * fs) + np.arange(N) / fs
    A, phi0, f = 1.3, 0.4, k * fs / N
    x64 = A * np.cos(phi0 + 2 * np.pi * f * t)
    x = x64.astype(np.float32)
    tol = 1e-6 * N
    for d in (0.0, 0.3, np.pi / 2, 2.0, np.pi):
        th = np.array([0.9, 123.0, phi0 + d, f, 0.0])                 # a1 = 123 must not matter (Eq. 6)
        assert abs(oracle.cor(x, fs, th) - 0.9 * A * (N / 2) * np.cos(d)) < tol
    # the model's frequency on another bin: orthogonal
    assert abs(oracle.cor(x, fs, np.array([1.0, 0.0, 0.1, (k + 3) * fs / N, 0.0]))) < tol


def test_hand_values_and_every_phase_term():
    # N = 4 at fs = 4: t = -0.5, -0.25, 0, 0.25
    x = np.array([1.0, -2.0, 0.5, 4.0], dtype=np.float32)
    th = np.array([2.0, 0.0, 0.0, 1.0, 0.0])                          # 2 cos(2 pi t): -2, 0, 2, 0
    assert abs(oracle.cor(x, 4.0, th) - (-2.0 * 1.0 + 2.0 * 0.5)) < 1e-14
    th = np.array([1.0, 0.0, np.pi / 2, 1.0, 0.0])                    # cos(pi/2 + 2 pi t) = -sin(2 pi t): 0, 1, 0, -1
    assert abs(oracle.cor(x, 4.0, th) - (-2.0 - 4.0)) < 1e-14
    # each phase coefficient enters with the sign and factor of Eq. 2-3 in Hz units
    rng = np.random.default_rng(0)
    N, fs = 64, 32.0
    t = -N / (2 * fs) + np.arange(N) / fs
    xs = rng.standard_normal(N).astype(np.float32)
    th = np.array([0.7, 0.0, 0.3, 3.1, -0.8, 1.7])
    ph = th[2] + 2 * np.pi * (th[3] * t + th[4] * t**2 / 2 + th[5] * t**3 / 6)
    assert abs(oracle.cor(xs, fs, th) - np.sum(xs.astype(np.float64) * th[0] * np.cos(ph))) < 1e-12


def test_symmetries():
    rng = np.random.default_rng(1)
    N, fs = 128, 64.0
    x = rng.standard_normal(N).astype(np.float32)
    th = np.array([0.8, 0.0, 0.5, 5.2, 0.7])
    c = oracle.cor(x, fs, th)
    assert abs(oracle.cor(-x, fs, th) + c) < 1e-13                    # odd in the data
    th2 = th.copy(); th2[0] *= 3
    assert abs(oracle.cor(x, fs, th2) - 3 * c) < 1e-12                # linear in A
    th3 = th.copy(); th3[2] += np.pi
    assert abs(oracle.cor(x, fs, th3) + c) < 1e-12                    # phase shift by pi flips the sign
    th4 = th.copy(); th4[2] += 2 * np.pi
    assert abs(oracle.cor(x, fs, th4) - c) < 1e-12
    # F_cor of the populations interface equals Eq. 5 of the correlation sum
    pop = np.stack([th, th2, th3]).astype(np.float32)[None]
    f = oracle.fitness(x[None], fs, pop, objective=1)
    for i in range(3):
        assert f[0, i] == oracle.fcor_of_cor(oracle.cor(x, fs, pop[0, i].astype(np.float64)))


def test_rss_and_cor_are_tied_by_the_expansion_of_the_square():
    """sum (x - s)^2 = sum x^2 - 2 cor + sum s^2 for the constant-amplitude model (a1 = 0)."""
    rng = np.random.default_rng(2)
    N, fs = 256, 128.0
    t = -N / (2 * fs) + np.arange(N) / fs
    x = rng.standard_normal(N).astype(np.float32)
    th = np.array([1.2, 0.0, -0.4, 11.3, 2.0])
    s = th[0] * np.cos(th[2] + 2 * np.pi * (th[3] * t + th[4] * t**2 / 2))
    lhs = oracle.rss(x, fs, th)
    rhs = np.sum(x.astype(np.float64) ** 2) - 2 * oracle.cor(x, fs, th) + np.sum(s**2)
    assert abs(lhs - rhs) < 1e-10 * lhs


def _ls_phase_fit(x, fs, t0, truth):
    t = t0 + np.arange(x.shape[0]) / fs
    xk = x.astype(np.float64)
    fun = lambda p: truth[0] * np.cos(p[0] + 2 * np.pi * (p[1] * t + p[2] * t * t / 2)) - xk
    sol = least_squares(fun, truth[2:5], method="lm", xtol=1e-14, ftol=1e-14, gtol=1e-14)
    return sol.x


@pytest.mark.parametrize("strategy", [6, 1])
def test_de_on_the_correlation_objective_finds_the_least_squares_phase(strategy):
    """Constant amplitude, zero-width (a0, a1) box: the maximiser of cor is, up to the slowly varying sum of s^2,
    the least-squares phase.  Strategy 6 is the paper's choice for Eq. 5."""
    wl = W.config0(cases=range(3), box="paper", a1_zero=True)
    lo, hi = wl.lo.copy(), wl.hi.copy()
    lo[:, 0] = hi[:, 0] = wl.truth[:, 0]
    lo[:, 1] = hi[:, 1] = 0.0
    r = oracle.fit_blocks(wl.x, wl.fs, lo, hi, NP=60, generations=300, F=0.5, CR=0.9, seed=23, strategy=strategy,
                          objective=1, want_pop=True, want_trace=True)
    for k in range(wl.B):
        ls = _ls_phase_fit(wl.x[k], wl.fs, wl.t0, wl.truth[k])
        d = r["best"][k, 2:5] - ls
        d[0] = (d[0] + np.pi) % (2 * np.pi) - np.pi
        # sum s^2 = a0^2 (N/2 + O(1)) moves the optimum by far less than the noise does
        assert abs(d[0]) < 2e-3 and abs(d[1]) < 1e-3 and abs(d[2]) < 2e-2
        assert r["best_rss"][k] == oracle.fcor_of_cor(oracle.cor(wl.x[k], wl.fs, r["best"][k]))
        assert np.all(np.diff(r["trace"][k]) <= 0)
        assert r["best_rss"][k] > 1 / np.pi
        assert (r["status"][k] & 2) == 0
        # collapsed population: every member's correlation within 1e-3 of the best
        c = np.array([oracle.cor(wl.x[k], wl.fs, p) for p in r["final_pop"][k]])
        assert np.ptp(c) < 1e-3 * c.max()
        # at the optimum cor ~ a0 A N/2
        assert abs(c.max() / (wl.truth[k, 0] ** 2 * wl.N / 2) - 1) < 0.05


def test_divergent_when_the_amplitude_is_free():
    """with a free amplitude "the objective function becomes divergent": a0 runs to its upper bound."""
    wl = W.config0(cases=[0], a1_zero=True)
    r = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=40, generations=200, seed=5, objective=1)
    assert abs(r["best"][0, 0] - wl.hi[0, 0]) <= 1e-6 * (wl.hi[0, 0] - wl.lo[0, 0])
    assert r["status"][0] & 1
