"""Pins of the oracle's Differential Evolution loop.

DE is a heuristic, so the oracle follows the algorithm step by step; it is pinned here by
(a) a pure-Python replay of single generations from the integer draws, (b) the closed form on
noiseless data, (c) brute force on a tiny block, (d) an independent Levenberg-Marquardt solve
(scipy) of the same least-squares problem, and (e) invariants of greedy selection.
"""
import numpy as np
from scipy.optimize import least_squares

import oracle
from paper_1906_10598_b200 import workloads as W


def _np_model(th, t):
    """Eq. 2 written in the paper's c-units (independent of the oracle's C code)."""
    c0, c1, c2 = th[2], 2 * np.pi * th[3], np.pi * th[4]
    c3 = np.pi / 3 * th[5] if len(th) > 5 else 0.0
    return (th[0] + th[1] * t) * np.cos(c0 + c1 * t + c2 * t**2 + c3 * t**3)


def _small_block(seed=3, N=200, fs=200.0, D=5):
    rng = np.random.default_rng(seed)
    t = -N / (2 * fs) + np.arange(N) / fs
    th = np.array([1.1, 0.05, 0.7, 23.0, 0.4, 0.8][:D])
    x = (_np_model(th, t) + 0.1 * rng.standard_normal(N)).astype(np.float32)
    return x[None, :], fs, th


def test_generation_zero_is_uniform_in_the_box():
    x, fs, th = _small_block()
    lo = (th - np.array([0.3, 0.1, 1.0, 2.0, 1.0]))[None, :]
    hi = (th + np.array([0.2, 0.2, 0.5, 3.0, 2.0]))[None, :]
    r = oracle.fit_blocks(x, fs, lo, hi, NP=9, generations=0, seed=77, block_index=[5], want_pop=True)
    for i in range(9):
        u = oracle.init_uniforms(77, 5, i, 5)
        assert np.array_equal(r["final_pop"][0, i], lo[0] + (hi[0] - lo[0]) * u)
        assert r["final_fit"][0, i] == oracle.rss(x[0], fs, r["final_pop"][0, i])
    ib = int(np.argmin(r["final_fit"][0]))
    assert np.array_equal(r["best"][0], r["final_pop"][0, ib])
    assert r["best_rss"][0] == r["final_fit"][0, ib]


def _replay(x, fs, lo, hi, NP, G, F, CR, seed, b, D):
    """Pure-Python DE/rand/1/bin, synchronous, reflect-then-clamp, accept on <=."""
    pop = np.array([lo + (hi - lo) * oracle.init_uniforms(seed, b, i, D) for i in range(NP)])
    fit = np.array([oracle.rss(x, fs, p) for p in pop])
    n_reflect = n_clamp = 0
    for g in range(1, G + 1):
        trial = pop.copy()
        for i in range(NP):
            r1, r2, r3, jrand, mask = oracle.de_draws(seed, b, g, i, NP, D, CR)
            for j in range(D):
                if (mask >> j) & 1:
                    u = pop[r1, j] + F * (pop[r2, j] - pop[r3, j])
                    if u < lo[j]:
                        u = 2 * lo[j] - u
                        n_reflect += 1
                    elif u > hi[j]:
                        u = 2 * hi[j] - u
                        n_reflect += 1
                    if u < lo[j] or u > hi[j]:
                        n_clamp += 1
                    u = min(max(u, lo[j]), hi[j])
                    trial[i, j] = u
        tfit = np.array([oracle.rss(x, fs, p) for p in trial])
        acc = tfit <= fit
        pop[acc] = trial[acc]
        fit[acc] = tfit[acc]
    return pop, fit, n_reflect, n_clamp


def test_generations_replayed_step_by_step():
    for D in (5, 6):
        x, fs, th = _small_block(D=D)
        half = np.array([0.3, 0.1, 1.0, 2.0, 1.0, 2.0][:D])
        lo, hi = th - half, th + half
        NP, G, F, CR, seed, b = 10, 6, 1.7, 0.6, 2024, 3
        pop, fit, n_reflect, n_clamp = _replay(x[0], fs, lo, hi, NP, G, F, CR, seed, b, D)
        assert n_reflect > 0 and n_clamp > 0          # both branches of the bound rule were exercised
        r = oracle.fit_blocks(x, fs, lo[None], hi[None], NP=NP, generations=G, F=F, CR=CR, seed=seed,
                              block_index=[b], want_pop=True)
        assert np.array_equal(r["final_pop"][0], pop)
        assert np.array_equal(r["final_fit"][0], fit)


def test_population_stays_in_box_and_zero_width_is_legal():
    x, fs, th = _small_block()
    lo = th - np.array([0.3, 0.0, 1.0, 2.0, 1.0])
    hi = th + np.array([0.3, 0.0, 1.0, 2.0, 1.0])        # a1 has a zero-width box
    r = oracle.fit_blocks(x, fs, lo[None], hi[None], NP=12, generations=40, F=1.9, CR=1.0, seed=1, want_pop=True,
                          want_trace=True)
    p = r["final_pop"][0]
    assert np.all(p >= lo) and np.all(p <= hi)
    assert np.all(p[:, 1] == th[1])
    assert np.all(np.diff(r["trace"][0]) <= 0)           # greedy selection never loses the best
    assert r["trace"][0, -1] == r["best_rss"][0]


def test_all_zero_width_box_ties_resolve_to_lowest_index():
    x, fs, th = _small_block()
    r = oracle.fit_blocks(x, fs, th[None], th[None], NP=5, generations=3, seed=9, want_pop=True)
    assert np.array_equal(r["best"][0], th)
    assert r["status"][0] == 0
    assert np.all(r["final_fit"][0] == r["final_fit"][0, 0])


def test_noiseless_recovers_truth():
    wl = W.config0(cases=range(2), noiseless=True)
    r = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=500, F=0.5, CR=0.9, seed=5)
    scale = np.maximum(np.abs(wl.truth), [1.0, 1.0, 1.0, 1.0, 1.0])
    assert np.all(np.abs(r["best"] - wl.truth) <= 1e-6 * scale)
    assert np.all(r["best_rss"] < 1e-9)
    assert np.all((r["status"] & 1) == 0)


def test_brute_force_grid_on_a_tiny_block():
    """N = 64, two free coordinates (phi0, f): the DE optimum agrees with an exhaustive grid to grid spacing."""
    rng = np.random.default_rng(8)
    N, fs = 64, 64.0
    t = -N / (2 * fs) + np.arange(N) / fs
    th = np.array([1.0, 0.0, 0.4, 9.3, 0.0])
    x = (_np_model(th, t) + 0.2 * rng.standard_normal(N)).astype(np.float32)
    lo = th.copy()
    hi = th.copy()
    lo[2], hi[2] = -1.0, 2.0
    lo[3], hi[3] = 8.8, 9.8
    n1, n2 = 601, 501
    p_grid = np.linspace(lo[2], hi[2], n1)
    f_grid = np.linspace(lo[3], hi[3], n2)
    P, Fq = np.meshgrid(p_grid, f_grid, indexing="ij")
    model = np.cos(P[..., None] + 2 * np.pi * Fq[..., None] * t)
    rss_grid = np.sum((x.astype(np.float64) - model) ** 2, axis=-1)
    i1, i2 = np.unravel_index(np.argmin(rss_grid), rss_grid.shape)
    r = oracle.fit_blocks(x[None], fs, lo[None], hi[None], NP=20, generations=150, seed=4)
    assert abs(r["best"][0, 2] - p_grid[i1]) <= (p_grid[1] - p_grid[0])
    assert abs(r["best"][0, 3] - f_grid[i2]) <= (f_grid[1] - f_grid[0])
    assert r["best_rss"][0] <= rss_grid[i1, i2] + 1e-12
    assert r["best_rss"][0] >= rss_grid[i1, i2] - 1e-3


def test_levenberg_marquardt_agreement_and_noise_floor():
    """The DE optimum on a noisy config-0 block is the least-squares optimum: scipy's LM started at the truth
    lands on the same point; RSS_best <= RSS(truth); RSS_best ~ (N - D) sigma^2."""
    wl = W.config0(cases=range(3), box="paper")
    r = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=500, F=0.5, CR=0.9, seed=11, want_pop=True)
    t = wl.t0 + np.arange(wl.N) / wl.fs
    for k in range(wl.B):
        xk = wl.x[k].astype(np.float64)
        sol = least_squares(lambda th: _np_model(th, t) - xk, wl.truth[k], method="lm", xtol=1e-14, ftol=1e-14,
                            gtol=1e-14)
        rss_lm = float(np.sum(sol.fun**2))
        assert abs(r["best_rss"][k] - rss_lm) <= 1e-9 * rss_lm
        d = r["best"][k] - sol.x
        d[2] = (d[2] + np.pi) % (2 * np.pi) - np.pi
        assert np.all(np.abs(d) <= 2e-5 * np.maximum(np.abs(sol.x), 1.0))
        assert r["best_rss"][k] <= oracle.rss(wl.x[k], wl.fs, wl.truth[k])
        s2 = wl.meta["sigma_per_block"][k] ** 2
        assert abs(r["best_rss"][k] - (wl.N - 5) * s2) < 4.5 * s2 * np.sqrt(2.0 * wl.N)
        assert (r["status"][k] & 2) == 0                       # collapsed
        assert np.ptp(r["final_pop"][k][:, 3]) < 1e-5          # population spread in f far below 1e-3 Hz


def test_paper_table4_settings_converge():
    """Table 4: F_XC = 0.5, CR_XC = 0.85, itermax = 200."""
    wl = W.config0(cases=[4])
    r = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=200, F=0.5, CR=0.85, seed=1)
    r2 = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=500, F=0.5, CR=0.9, seed=2)
    assert abs(r["best_rss"][0] - r2["best_rss"][0]) < 1e-6 * r2["best_rss"][0]


def test_status_face_bit_when_optimum_is_outside_the_box():
    wl = W.config0(cases=[1])
    lo, hi = wl.lo.copy(), wl.hi.copy()
    lo[0, 3] = wl.truth[0, 3] + 0.05           # the box for f excludes the truth: best must sit on the face
    hi[0, 3] = wl.truth[0, 3] + 0.5
    r = oracle.fit_blocks(wl.x, wl.fs, lo, hi, NP=40, generations=300, seed=3)
    assert r["status"][0] & 1
    assert abs(r["best"][0, 3] - lo[0, 3]) <= 1e-6 * (hi[0, 3] - lo[0, 3])


def test_not_collapsed_bit_early():
    wl = W.config0(cases=[2])
    r = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=30, generations=2, seed=3)
    assert r["status"][0] & 2


def test_block_index_selects_the_random_stream():
    wl = W.config0(cases=range(2))
    a = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=10, generations=3, seed=3, want_pop=True)
    b = oracle.fit_blocks(wl.x[1:], wl.fs, wl.lo[1:], wl.hi[1:], NP=10, generations=3, seed=3, block_index=[1],
                          want_pop=True)
    assert np.array_equal(a["final_pop"][1], b["final_pop"][0])
