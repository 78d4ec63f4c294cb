"""Pins of the oracle's signal model and chi^2 objective (Eq. 2-4).

Checked against values the mathematics fixes: hand values at phases that are multiples of pi/2,
the paper's own c0..c5 parameterisation written out independently, the noiseless closed form
RSS(theta_true) = 0, and the expectation "sum of noise power".
"""
import numpy as np

import oracle
from paper_1906_10598_b200 import workloads as W


def _times(N, fs):
    return -N / (2.0 * fs) + np.arange(N) / fs


def test_time_grid_and_hand_values_quarter_rate():
    """N = 8, fs = 8 Hz: t_n = (n - 4)/8.  f = fs/4 = 2 Hz gives phase (pi/2)(n - 4): cos = +1, 0, -1, 0 ..."""
    N, fs = 8, 8.0
    a0, a1 = 2.0, 0.5
    th = [a0, a1, 0.0, 2.0, 0.0]
    t = _times(N, fs)
    cosv = np.array([1.0, 0.0, -1.0, 0.0, 1.0, 0.0, -1.0, 0.0])       # m = -4 .. 3, cos(pi m / 2)
    for n in range(N):
        assert abs(oracle.model(th, t[n]) - (a0 + a1 * t[n]) * cosv[n]) < 1e-14
    # RSS against x = 0 keeps only the even samples: sum (a0 + a1 t)^2 over m = -4, -2, 0, 2
    expect = sum((a0 + a1 * (m / 8.0)) ** 2 for m in (-4, -2, 0, 2))
    assert abs(oracle.rss(np.zeros(N, np.float32), fs, th) - expect) < 1e-12
    # sample N/2 sits at t = 0 (left-closed block [-T/2, T/2))
    x = np.zeros(N, np.float32)
    x[N // 2] = a0
    assert abs(oracle.rss(x, fs, th) - (expect - a0**2)) < 1e-12


def test_sign_of_every_phase_term():
    """With phi0 = pi/2 the model is -A sin(rest): odd in the sign of f t and fddot t^3, so a wrong sign or a
    swapped coefficient shows up as a sign flip of exact +-1 values."""
    fs = 8.0
    # f = 2 Hz: rest = (pi/2) m -> s(m=+1) = A cos(pi) = -A, s(m=-1) = A cos(0) = +A
    th = [1.0, 0.0, np.pi / 2, 2.0, 0.0]
    assert abs(oracle.model(th, 1 / fs) + 1.0) < 1e-14
    assert abs(oracle.model(th, -1 / fs) - 1.0) < 1e-14
    # fdot: t^2/2 term, even in t.  fdot = 64: fdot t^2/2 = m^2/2 cycles -> cos = +1 (m even), -1 (m odd)
    th = [1.0, 0.0, 0.0, 0.0, 64.0]
    for m in range(-4, 4):
        assert abs(oracle.model(th, m / fs) - (1.0 if m % 2 == 0 else -1.0)) < 1e-12
    # fdot with phi0 = pi/2 and a quarter cycle: fdot = 32 -> m^2/4 cycles; m = +-1 -> cos(pi/2 + pi/2) = -1
    th = [1.0, 0.0, np.pi / 2, 0.0, 32.0]
    assert abs(oracle.model(th, 1 / fs) + 1.0) < 1e-12
    assert abs(oracle.model(th, -1 / fs) + 1.0) < 1e-12
    # fddot: t^3/6 term, odd in t.  fddot = 768: fddot t^3/6 = m^3/4 cycles; with phi0 = pi/2:
    # m = +1 -> cos(pi) = -1, m = -1 -> cos(0) = +1, m = 2 -> cos(pi/2 + 4 pi) = 0
    th = [1.0, 0.0, np.pi / 2, 0.0, 0.0, 768.0]
    assert abs(oracle.model(th, 1 / fs) + 1.0) < 1e-12
    assert abs(oracle.model(th, -1 / fs) - 1.0) < 1e-12
    assert abs(oracle.model(th, 2 / fs)) < 1e-12
    # D = 5 ignores a sixth number
    assert oracle.model([1.0, 0.0, 0.3, 1.0, 0.2], 0.37) == oracle.model([1.0, 0.0, 0.3, 1.0, 0.2, 0.0], 0.37)


def test_amplitude_slope():
    # phi = 0 everywhere: s = a0 + a1 t
    th = [1.5, -0.25, 0.0, 0.0, 0.0]
    for t in (-0.5, -0.125, 0.0, 0.25):
        assert abs(oracle.model(th, t) - (1.5 - 0.25 * t)) < 1e-15


def test_model_equals_paper_parameterisation():
    """Eq. 2 in the paper's own units: s = (c4 + c5 t) cos(c0 + c1 t + c2 t^2 + c3 t^3) with
    c0 = phi0, c1 = 2 pi f, c2 = pi fdot, c3 = (pi/3) fddot, c4 = a0, c5 = a1 (Eq. 3: c_i = phi^(i)(0)/i!)."""
    rng = np.random.default_rng(5)
    for _ in range(50):
        a0, a1 = rng.uniform(0.5, 1.5), rng.uniform(-0.1, 0.1)
        phi0, f, fdot, fddot = rng.uniform(-3, 3), rng.uniform(50, 200), rng.uniform(-1, 1), rng.uniform(-5, 5)
        c = [phi0, 2 * np.pi * f, np.pi * fdot, np.pi / 3 * fddot, a0, a1]
        t = rng.uniform(-0.5, 0.5)
        s = (c[4] + c[5] * t) * np.cos(c[0] + c[1] * t + c[2] * t**2 + c[3] * t**3)
        assert abs(oracle.model([a0, a1, phi0, f, fdot, fddot], t) - s) < 1e-10
        # Eq. 3 check by finite differences of the phase: phi'(0) = c1, phi''(0) = 2 c2, phi'''(0) = 6 c3
        h = 1e-3

        def ph(tt):
            return phi0 + 2 * np.pi * (f * tt + fdot * tt**2 / 2 + fddot * tt**3 / 6)

        d1 = (ph(h) - ph(-h)) / (2 * h)
        assert abs(d1 - c[1]) < 1e-3 * abs(c[1]) * 1e-3 + 1e-4


def test_noiseless_rss_is_zero_at_truth():
    """Closed form: on a noiseless signal RSS(theta_true) = 0 up to the fp32 rounding of the samples,
    bounded by N (2^-24 A)^2 (SURVEY 8(c) fitness pin (i))."""
    wl = W.config0(cases=range(8), noiseless=True)
    for k in range(wl.B):
        r = oracle.rss(wl.x[k], wl.fs, wl.truth[k])
        amax = abs(wl.truth[k, 0]) + 0.5 * abs(wl.truth[k, 1])
        assert 0.0 <= r <= wl.N * (2.0**-24 * amax) ** 2
    # and it is not zero a little away from the truth
    th = wl.truth[0].copy()
    th[3] += 0.01
    assert oracle.rss(wl.x[0], wl.fs, th) > 1e-3


def test_noisy_rss_at_truth_is_noise_power():
    """the chi^2 objective converges to the summed noise power: E[RSS(theta_true)] = N sigma^2,
    variance 2 N sigma^4."""
    wl = W.config0(cases=range(32))
    z = []
    for k in range(wl.B):
        s2 = wl.meta["sigma_per_block"][k] ** 2
        r = oracle.rss(wl.x[k], wl.fs, wl.truth[k])
        z.append((r - wl.N * s2) / (s2 * np.sqrt(2.0 * wl.N)))
    z = np.array(z)
    assert np.all(np.abs(z) < 4.5)
    assert abs(z.mean()) < 4.0 / np.sqrt(len(z))


def test_pure_noise_expectation():
    """x = noise only: E[RSS(theta)] = N sigma^2 + sum s(theta)^2 (SURVEY fitness pin (iii))."""
    rng = np.random.default_rng(11)
    N, fs, sig = 4000, 4000.0, 0.7
    th = [1.2, 0.05, 0.4, 333.0, 0.3]
    t = _times(N, fs)
    s2 = float(np.sum(((th[0] + th[1] * t) * np.cos(th[2] + 2 * np.pi * (th[3] * t + th[4] * t * t / 2))) ** 2))
    vals = []
    for _ in range(40):
        x = (sig * rng.standard_normal(N)).astype(np.float32)
        vals.append(oracle.rss(x, fs, th))
    mean = np.mean(vals)
    sd = np.sqrt(2 * N * sig**4 + 4 * sig**2 * s2) / np.sqrt(40)
    assert abs(mean - (N * sig**2 + s2)) < 4.5 * sd


def test_fitness_batch_matches_rss_and_promotes_fp32():
    wl = W.config0(cases=range(3))
    rng = np.random.default_rng(2)
    NP = 7
    pop = (wl.lo[:, None, :] + (wl.hi - wl.lo)[:, None, :] * rng.uniform(size=(wl.B, NP, 5))).astype(np.float32)
    fit = oracle.fitness(wl.x, wl.fs, pop)
    assert fit.shape == (wl.B, NP) and fit.dtype == np.float64
    for b in range(wl.B):
        for i in range(NP):
            assert fit[b, i] == oracle.rss(wl.x[b], wl.fs, pop[b, i].astype(np.float64))


def test_t0_argument_shifts_the_grid():
    wl = W.config0(cases=[0], noiseless=True)
    th = wl.truth[0]
    # evaluating with t0 shifted by one sample must equal evaluating the shifted-parameter signal:
    # it is not ~0 any more
    r0 = oracle.rss(wl.x[0], wl.fs, th)
    r1 = oracle.rss(wl.x[0], wl.fs, th, t0=wl.t0 + 1.0 / wl.fs)
    assert r0 < 1e-10 and r1 > 1.0
