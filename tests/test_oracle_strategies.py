"""Pins of the oracle's six mutation strategies ("six kind of mutation operations strategies ... the
third is the best choice for objective function Eq. 4 and the sixth for Eq. 5", Table 4 :220; reading R21).

The paper never defines the strategies, so there is no printed value to compare with.  The pins are what the
definitions themselves fix: geometric invariants of every trial vector (which point it starts from, along which
direction it moves, by how much), the distribution of the random scale factors, limiting cases (F = 0, F = 1),
and that every strategy reaches the optimum an independent solver (scipy Levenberg-Marquardt) finds.
"""
import numpy as np
import pytest
from scipy.optimize import least_squares

import oracle
from paper_1906_10598_b200 import workloads as W

SEED = 424242
D = 5
NP = 12


def _population(rng):
    pop = rng.uniform(-1.0, 1.0, size=(NP, D))
    fit = rng.uniform(1.0, 2.0, size=NP)
    return pop, int(np.argmin(fit))


def _wide_box():
    return np.full(D, -1e6), np.full(D, 1e6)


def _trial(pop, ibest, strategy, *, F=0.5, CR=1.0, g=1, i=0, b=0, lo=None, hi=None):
    wlo, whi = _wide_box()
    return oracle.de_trial(pop, ibest, wlo if lo is None else lo, whi if hi is None else hi, b=b, g=g, i=i, F=F, CR=CR,
                           seed=SEED, strategy=strategy)


def test_aux_uniforms_are_philox_words_of_slots_3_and_4():
    jit, uvec, ugen = oracle.aux_uniforms(SEED, 7, 3, 5)
    key = [SEED & 0xFFFFFFFF, SEED >> 32]
    w3 = oracle.philox4x32_10([3, 5, 3, 7], key)
    w4 = oracle.philox4x32_10([4, 5, 3, 7], key)
    wg = oracle.philox4x32_10([3, 0xFFFFFFFF, 3, 7], key)
    assert np.array_equal(jit[:4], (w3 >> 8) / 2.0**24)
    assert np.array_equal(jit[4:], (w4 >> 8) / 2.0**24)
    assert uvec == (int(w3[0]) >> 8) / 2.0**24
    assert ugen == (int(wg[0]) >> 8) / 2.0**24
    # the per-generation number does not depend on the candidate, the per-vector one does
    _, uvec2, ugen2 = oracle.aux_uniforms(SEED, 7, 3, 6)
    assert ugen2 == ugen and uvec2 != uvec


def test_strategy1_is_rand1():
    rng = np.random.default_rng(0)
    pop, ib = _population(rng)
    for i in range(NP):
        r1, r2, r3, _, _ = oracle.de_draws(SEED, 0, 1, i, NP, D, 1.0)
        v = _trial(pop, ib, 1, i=i)
        assert np.array_equal(v, pop[r1] + 0.5 * (pop[r2] - pop[r3]))


def test_strategy2_local_to_best_limits():
    rng = np.random.default_rng(1)
    pop, ib = _population(rng)
    for i in range(NP):
        _, r2, r3, _, _ = oracle.de_draws(SEED, 0, 1, i, NP, D, 1.0)
        # F = 0: the trial is the parent itself
        assert np.array_equal(_trial(pop, ib, 2, F=0.0, i=i), pop[i])
        # F = 1: x_i + (x_best - x_i) + (x_r2 - x_r3) = x_best + (x_r2 - x_r3) up to rounding
        v = _trial(pop, ib, 2, F=1.0, i=i)
        assert np.allclose(v, pop[ib] + (pop[r2] - pop[r3]), rtol=0, atol=1e-14)
        # general F: the displacement from the parent is F (x_best - x_i) + F (x_r2 - x_r3)
        v = _trial(pop, ib, 2, F=0.3, i=i)
        assert np.allclose(v - pop[i], 0.3 * (pop[ib] - pop[i]) + 0.3 * (pop[r2] - pop[r3]), rtol=0, atol=1e-14)
    # the best member itself only moves along the difference vector
    _, r2, r3, _, _ = oracle.de_draws(SEED, 0, 1, ib, NP, D, 1.0)
    assert np.allclose(_trial(pop, ib, 2, F=0.7, i=ib) - pop[ib], 0.7 * (pop[r2] - pop[r3]), rtol=0, atol=1e-14)


def test_strategy3_best1_with_jitter():
    rng = np.random.default_rng(2)
    pop, ib = _population(rng)
    ratios = []
    for g in range(1, 40):
        for i in range(NP):
            _, r2, r3, _, _ = oracle.de_draws(SEED, 0, g, i, NP, D, 1.0)
            v = _trial(pop, ib, 3, F=0.5, g=g, i=i)
            ratio = (v - pop[ib]) / (pop[r2] - pop[r3])       # per-coordinate scale factor F + 0.0001 rand_j
            assert np.all(ratio >= 0.5 - 1e-12) and np.all(ratio < 0.5001 + 1e-12)
            assert len(np.unique(np.round(ratio, 12))) > 1      # jitter differs between coordinates
            ratios.append(ratio)
            # F = 0 leaves only the jitter: |v - x_best| < 1e-4 |x_r2 - x_r3|
            v0 = _trial(pop, ib, 3, F=0.0, g=g, i=i)
            assert np.all(np.abs(v0 - pop[ib]) <= 1.0001e-4 * np.abs(pop[r2] - pop[r3]))
    u = (np.concatenate(ratios) - 0.5) / 1e-4                   # the jitter numbers are uniform in [0, 1)
    assert abs(u.mean() - 0.5) < 4 * np.sqrt(1 / 12 / u.size)
    assert abs(u.var() - 1 / 12) < 0.01


@pytest.mark.parametrize("strategy", [4, 5])
def test_dither_strategies(strategy):
    rng = np.random.default_rng(3)
    pop, ib = _population(rng)
    F = 0.3
    per_gen = []
    for g in range(1, 60):
        scales = []
        for i in range(NP):
            r1, r2, r3, _, _ = oracle.de_draws(SEED, 0, g, i, NP, D, 1.0)
            v = _trial(pop, ib, strategy, F=F, g=g, i=i)
            ratio = (v - pop[r1]) / (pop[r2] - pop[r3])
            assert np.allclose(ratio, ratio[0], rtol=0, atol=1e-10)   # one scale factor for the whole vector
            assert F - 1e-10 <= ratio[0] < 1.0 + 1e-10                  # F + (1 - F) rand in [F, 1)
            scales.append(ratio[0])
        scales = np.array(scales)
        if strategy == 5:
            assert np.allclose(scales, scales[0], rtol=0, atol=1e-10)   # the same for every vector of a generation
        else:
            assert np.ptp(scales) > 1e-3                                # differs between vectors
        per_gen.append(scales)
    allv = np.concatenate(per_gen) if strategy == 4 else np.array([s[0] for s in per_gen])
    assert np.ptp(allv) > 0.3                                           # and between generations
    # mean of F + (1 - F) U(0,1) is (1 + F)/2
    assert abs(allv.mean() - (1 + F) / 2) < 4 * (1 - F) * np.sqrt(1 / 12 / allv.size)


def test_strategy6_either_or():
    rng = np.random.default_rng(4)
    pop, ib = _population(rng)
    F = 0.4
    K = 0.5 * (F + 1.0)
    n_de = n_rec = 0
    for g in range(1, 80):
        for i in range(NP):
            r1, r2, r3, _, _ = oracle.de_draws(SEED, 0, g, i, NP, D, 1.0)
            v = _trial(pop, ib, 6, F=F, g=g, i=i)
            de = pop[r1] + F * (pop[r2] - pop[r3])
            rec = pop[r1] + K * (pop[r2] + pop[r3] - 2 * pop[r1])
            is_de = np.allclose(v, de, rtol=0, atol=1e-14)
            is_rec = np.allclose(v, rec, rtol=0, atol=1e-14)
            assert is_de != is_rec                                      # the whole vector takes one branch
            _, uvec, _ = oracle.aux_uniforms(SEED, 0, g, i)
            assert is_de == (uvec < 0.5)
            n_de += is_de
            n_rec += is_rec
    n = n_de + n_rec
    assert abs(n_de - n / 2) < 4 * np.sqrt(n / 4)                       # p = 1/2


@pytest.mark.parametrize("strategy", [1, 2, 3, 4, 5, 6])
def test_crossover_and_bounds_are_shared_by_every_strategy(strategy):
    rng = np.random.default_rng(5)
    pop, ib = _population(rng)
    lo, hi = np.full(D, -1.0), np.full(D, 1.0)
    n_kept = 0
    for g in range(1, 30):
        for i in range(NP):
            *_, mask = oracle.de_draws(SEED, 2, g, i, NP, D, 0.5)
            v = _trial(pop, ib, strategy, F=1.9, CR=0.5, g=g, i=i, b=2, lo=lo, hi=hi)
            free = _trial(pop, ib, strategy, F=1.9, CR=0.5, g=g, i=i, b=2)
            assert np.all(v >= lo) and np.all(v <= hi)
            for j in range(D):
                if not (mask >> j) & 1:
                    assert v[j] == pop[i, j]
                    n_kept += 1
                else:
                    u = free[j]
                    if u < lo[j]:
                        u = 2 * lo[j] - u
                    elif u > hi[j]:
                        u = 2 * hi[j] - u
                    assert v[j] == min(max(u, lo[j]), hi[j])
    assert n_kept > 100


def _np_model(th, t):
    return (th[0] + th[1] * t) * np.cos(th[2] + 2 * np.pi * (th[3] * t + th[4] * t * t / 2))


@pytest.mark.parametrize("strategy", [2, 3, 4, 5, 6])
def test_every_strategy_reaches_the_least_squares_optimum(strategy):
    # best/1 trades robustness for speed: on this wide box it stalls with F = 0.5 (premature convergence, the reason
    # the paper re-searches doubtful blocks) and reaches the optimum on every block with F = 0.7
    wl = W.config0(cases=range(2), box="paper")
    F = {3: 0.7, 5: 0.3}.get(strategy, 0.5)
    r = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=400, F=F, CR=0.9, seed=17, strategy=strategy,
                          want_trace=True)
    t = wl.t0 + np.arange(wl.N) / wl.fs
    for k in range(wl.B):
        xk = wl.x[k].astype(np.float64)
        sol = least_squares(lambda th: _np_model(th, t) - xk, wl.truth[k], method="lm", xtol=1e-14, ftol=1e-14,
                            gtol=1e-14)
        rss_lm = float(np.sum(sol.fun**2))
        assert abs(r["best_rss"][k] - rss_lm) <= 1e-8 * rss_lm
        assert np.all(np.diff(r["trace"][k]) <= 0)
    # noiseless data: the truth is recovered
    wl0 = W.config0(cases=[5], noiseless=True)
    r0 = oracle.fit_blocks(wl0.x, wl0.fs, wl0.lo, wl0.hi, NP=60, generations=500, F=F, CR=0.9, seed=3, strategy=strategy)
    assert np.all(np.abs(r0["best"] - wl0.truth) <= 1e-6 * np.maximum(np.abs(wl0.truth), 1.0))


def test_best1_converges_faster_than_rand1():
    """The reason the paper gives for picking a best-guided strategy with itermax = 200."""
    wl = W.config0(cases=range(4))
    a = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=120, F=0.5, CR=0.85, seed=5, strategy=1,
                          want_trace=True)
    b = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=120, F=0.5, CR=0.85, seed=5, strategy=3,
                          want_trace=True)
    # generation at which the best member is within 1e-6 of its final value
    def settle(tr):
        return int(np.argmax(tr <= tr[-1] * (1 + 1e-6)))
    ga = [settle(a["trace"][k]) for k in range(wl.B)]
    gb = [settle(b["trace"][k]) for k in range(wl.B)]
    assert np.mean(gb) < np.mean(ga)


def test_invalid_strategy_is_rejected():
    wl = W.config0(cases=[0])
    with pytest.raises(ValueError):
        oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=10, generations=1, strategy=7)
