"""Pins of the oracle's run-time ranges and re-search of doubtful blocks (reading R25).

What fixes it: the flag rule on hand-made border residuals; the extrapolation formulas on an exact polynomial-phase
track, where block n's Taylor polynomial IS block n+k's (closed form: F^n(kT) = f^{n+k}, F'^n(kT) = fdot^{n+k}), and the
paper's own interval [phi'^n(T/2), phi'^n(3T/2)] for k = 1; a scenario with deliberately wrong ranges that the first fit
cannot solve and one re-search repairs; a block without signal, abandoned after three attempts.
"""
import numpy as np

import oracle
from paper_1906_10598_b200 import workloads as W


def _per_block(bad_borders, B):
    pb = np.zeros((B, 10))
    for j in bad_borders:
        pb[j, 8] = 2.0
    pb[-1, 8:] = np.nan
    return pb


def test_flag_rule():
    B = 8
    f = lambda bad: list(np.nonzero(oracle.doubtful_blocks(_per_block(bad, B), 0.5, 0.5))[0])
    assert f([]) == []
    assert f([2, 3]) == [3]                 # an isolated wrong block spoils both of its borders
    assert f([2, 3, 4]) == [3, 4]           # two adjacent wrong blocks
    assert f([0]) == [0]                    # the first block has one border only
    assert f([6]) == [7]                    # so has the last
    assert f([0, 1]) == [0, 1]              # block 1 wrong: block 0 cannot be told apart and is searched again too
    # the frequency residual alone also marks a border (column 9 is rad/s, the threshold is in Hz)
    pb = _per_block([], B)
    pb[2, 9] = 2 * np.pi * 0.6
    pb[3, 9] = -2 * np.pi * 0.6
    assert list(np.nonzero(oracle.doubtful_blocks(pb, 0.5, 0.5))[0]) == [3]
    pb[3, 9] = -2 * np.pi * 0.4
    assert not oracle.doubtful_blocks(pb, 0.5, 0.5).any()
    assert not oracle.doubtful_blocks(np.full((1, 10), np.nan), 0.5, 0.5).any()      # a single block has no border


def test_extrapolation_is_exact_on_a_polynomial_phase():
    """phi(t) cubic in absolute time: every block's (f, fdot, fddot) is the same polynomial re-expanded, so block n
    predicts block n + k exactly; the paper's interval for k = 1 is [F^n(T/2), F^n(3T/2)]."""
    T, B = 2.0, 7
    f0, f1, f2 = 1000.0, 3.0, 0.4                      # f(t) = f0 + f1 t + f2 t^2 / 2
    tc = (np.arange(B) + 0.5) * T
    best = np.stack([np.ones(B), np.zeros(B), np.zeros(B), f0 + f1 * tc + f2 * tc**2 / 2, f1 + f2 * tc, np.full(B, f2)], axis=1)
    lo0, hi0 = best - 1.0, best + 1.0
    flags = np.zeros(B, dtype=bool)
    flags[3] = True
    lo, hi = oracle.extrapolated_box(3, flags, best, lo0[3], hi0[3], T, 1.0, 2.0, 0.0, 0.0, 0.1)
    Fn = lambda t: best[2, 3] + best[2, 4] * t + best[2, 5] * t * t / 2
    assert np.allclose([lo[3], hi[3]], [Fn(T / 2), Fn(3 * T / 2)], rtol=0, atol=1e-12)        # the paper's interval
    assert lo[3] <= best[3, 3] <= hi[3] and lo[4] <= best[3, 4] <= hi[4]
    assert abs(0.5 * (lo[4] + hi[4]) - best[3, 4]) < 1e-12                                   # F'^n(T) = fdot^{n+1}
    assert abs(0.5 * (lo[3] + hi[3]) - best[3, 3] - f2 * T * T / 8) < 1e-12                  # midpoint of a parabola's chord
    assert np.allclose([lo[0], hi[0]], [0.9, 1.1]) and np.allclose([lo[2], hi[2]], [-np.pi, np.pi])
    assert lo[1] == lo0[3, 1] and hi[5] == hi0[3, 5]                                         # a1, fddot keep their ranges
    # nearest trusted block: with 2 and 3 doubtful block 3 takes block 4 (distance 1, backwards, k = -1), block 2 takes 1
    flags[2] = True
    lo, hi = oracle.extrapolated_box(3, flags, best, lo0[3], hi0[3], T, 1.0, 2.0, 0.0, 0.0, 0.1)
    Fn = lambda t: best[4, 3] + best[4, 4] * t + best[4, 5] * t * t / 2
    assert np.allclose(sorted([lo[3], hi[3]]), sorted([Fn(-T / 2), Fn(-3 * T / 2)]), rtol=0, atol=1e-12)
    assert lo[3] <= best[3, 3] <= hi[3]
    # floors and the enlargement of later attempts
    lo, hi = oracle.extrapolated_box(3, flags, best, lo0[3], hi0[3], T, 4.0, 2.0, 50.0, 7.0, 0.1)
    assert abs((hi[3] - lo[3]) / 2 - 200.0) < 1e-9 and abs((hi[4] - lo[4]) / 2 - 28.0) < 1e-9
    assert np.allclose([lo[0], hi[0]], [0.6, 1.4])
    # nobody trusted: the own box is widened about its centre
    lo, hi = oracle.extrapolated_box(3, np.ones(B, dtype=bool), best, lo0[3], hi0[3], T, 1.0, 2.0, 0.0, 0.0, 0.1)
    assert np.allclose(lo, best[3] - 2.0) and np.allclose(hi, best[3] + 2.0)


def _scenario():
    wl = W.config1(blocks=range(8), generations=150, NP=40)
    lo, hi = wl.lo.copy(), wl.hi.copy()
    for b in (2, 5):                                   # ranges that do not cover the true frequency
        lo[b, 3] = wl.truth[b, 3] + 8.0
        hi[b, 3] = wl.truth[b, 3] + 30.0
    return wl, lo, hi


def test_wrong_ranges_are_found_and_repaired_by_one_re_search():
    wl, lo, hi = _scenario()
    good = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=40, generations=150, seed=5)
    first = oracle.fit_blocks(wl.x, wl.fs, lo, hi, NP=40, generations=150, seed=5)
    assert np.all(np.abs(first["best"][[2, 5], 3] - wl.truth[[2, 5], 3]) > 7.0)
    r = oracle.refit_doubtful(wl.x, wl.fs, lo, hi, first["best"], first["best_rss"], first["status"], NP=40,
                              generations=150, seed=5, phi_tol=0.5, F_tol=0.5, f_floor=2.0, fdot_floor=2.0)
    assert [list(np.nonzero(f)[0]) for f in r["flags_per_attempt"]] == [[2, 5], []]
    assert list(r["attempts"]) == [0, 0, 1, 0, 0, 1, 0, 0]
    assert not np.any(r["status"] & 4)
    assert np.array_equal(r["best"][[0, 1, 3, 4, 6, 7]], first["best"][[0, 1, 3, 4, 6, 7]])      # trusted blocks are untouched
    d = r["best"][[2, 5]] - good["best"][[2, 5]]
    assert np.max(np.abs((d[:, 2] + np.pi) % (2 * np.pi) - np.pi)) < 5e-3 and np.max(np.abs(d[:, 3])) < 1e-3
    assert np.all(r["lo"][[2, 5], 3] <= wl.truth[[2, 5], 3]) and np.all(wl.truth[[2, 5], 3] <= r["hi"][[2, 5], 3])
    # the re-search used another random stream
    again = oracle.fit_blocks(wl.x[[2]], wl.fs, r["lo"][[2]], r["hi"][[2]], NP=40, generations=150, seed=5, block_index=[2])
    assert not np.array_equal(again["best"], r["best"][[2]])
    again = oracle.fit_blocks(wl.x[[2]], wl.fs, r["lo"][[2]], r["hi"][[2]], NP=40, generations=150,
                              seed=(5 + 0x9E3779B97F4A7C15) % 2**64, block_index=[2])
    assert np.array_equal(again["best"], r["best"][[2]])


def test_a_block_without_signal_is_abandoned_after_three_attempts():
    wl = W.config1(blocks=range(6), generations=100, NP=30)
    x = wl.x.copy()
    rng = np.random.default_rng(1)
    x[3] = (wl.sigma * rng.standard_normal(wl.N)).astype(np.float32)          # the carrier drops out in block 3
    first = oracle.fit_blocks(x, wl.fs, wl.lo, wl.hi, NP=30, generations=100, seed=2)
    r = oracle.refit_doubtful(x, wl.fs, wl.lo, wl.hi, first["best"], first["best_rss"], first["status"], NP=30,
                              generations=100, seed=2, phi_tol=0.3, F_tol=0.2, f_floor=2.0, fdot_floor=2.0)
    assert r["attempts"][3] == 3 and r["status"][3] & 4
    assert len(r["flags_per_attempt"]) == 4 and all(f[3] for f in r["flags_per_attempt"])
    others = [0, 1, 2, 4, 5]
    assert not np.any(r["status"][others] & 4) and np.all(r["attempts"][others] == 0)
    # the range of block 3 grew by `grow` per attempt
    assert abs((r["hi"][3, 3] - r["lo"][3, 3]) / 2 - 4 * max(2.0, abs(first["best"][2, 4]) * wl.T / 2)) < 1e-6
