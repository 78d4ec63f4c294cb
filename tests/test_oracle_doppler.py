"""Pins of the oracle's Doppler products (PAPER.md:228-246 Eq. 7-8, :343-352 Eq. 16-17, :376-379 Eq. 19).

The worked example the paper prints (Appendix A; fixture tests/golden/appendix_a.txt)
pins Eq. 7, 8 and 17 to the paper's own numbers; invariants and a globally polynomial phase pin the rest.
"""
import os

import numpy as np

import oracle

T_MEX = 2.0


def _read_appendix(golden_dir):
    blocks, borders, edges = [], [], {}
    with open(os.path.join(golden_dir, "appendix_a.txt")) as fh:
        for line in fh:
            tok = line.split()
            if not tok or tok[0].startswith("#"):
                continue
            if tok[0] == "BLOCK":
                blocks.append([float(v) for v in tok[1:]])
            elif tok[0] == "BORDER":
                borders.append([float(v) for v in tok[1:]])
            else:
                edges[tok[0]] = [float(v) for v in tok[1:]]
    return np.array(blocks), np.array(borders), edges


def _theta_from_paper_units(row):
    """BLOCK row (sec, c0, c1, c2, c3, c4, c5, total) -> (a0, a1, phi0, f, fdot, fddot) by Eq. 3's mapping."""
    _, c0, c1, c2, c3, c4, c5, _ = row
    if np.isnan(c0):
        c0 = 0.0
    return [c4, c5, c0, c1 / (2 * np.pi), c2 / np.pi, 3.0 * c3 / np.pi]


def test_appendix_a_worked_example(golden_dir):
    blocks, borders, edges = _read_appendix(golden_dir)
    assert blocks.shape == (11, 8) and borders.shape == (10, 5)
    best = np.array([_theta_from_paper_units(r) for r in blocks])
    per_block, total, _ = oracle.doppler_products(best, T_MEX)
    # column 8: total_phase over the block = phi(T/2) - phi(-T/2), printed to 0.001 rad
    assert np.all(np.abs(per_block[:, 7] - blocks[:, 7]) <= 1.5e-3)
    for k, (sec, ph_l, f_l, ph_r, f_r) in enumerate(borders):
        assert sec == blocks[k, 0] + 1 == blocks[k + 1, 0] - 1
        # frequency at the border from the left block at +T/2 and from the right block at -T/2 (Eq. 8);
        # c3 is printed with 3 decimals, i.e. +-0.0005 rad/s^3, worth +-0.0015 rad/s at the border
        assert abs(per_block[k, 6] - f_l) <= 3e-3
        assert abs(per_block[k + 1, 5] - f_r) <= 3e-3
        # phase mod 2 pi at the border; c0 printed to 0.001 rad
        if k > 0:                                 # c0 of the first block is not printed
            d = (per_block[k, 4] - ph_l + np.pi) % (2 * np.pi) - np.pi
            assert abs(d) <= 2.5e-3
        d = (per_block[k + 1, 3] - ph_r + np.pi) % (2 * np.pi) - np.pi
        assert abs(d) <= 2.5e-3
    assert abs(per_block[0, 5] - edges["EDGE_LEFT"][2]) <= 3e-3
    assert abs(per_block[-1, 6] - edges["EDGE_RIGHT"][2]) <= 3e-3
    d = (per_block[-1, 4] - edges["EDGE_RIGHT"][1] + np.pi) % (2 * np.pi) - np.pi
    assert abs(d) <= 2.5e-3
    # phases are reported in [0, 2 pi) as the paper prints them
    assert np.all((per_block[:, 3:5] >= 0) & (per_block[:, 3:5] < 2 * np.pi))
    # continuity residuals (Eq. 8): the paper says continuity "can be confirmed" at the 50 mrad noise level
    bd = per_block[1:-1, 8]
    assert np.all(np.abs(bd) < 0.05)
    printed = (borders[1:, 3] - borders[1:, 1] + np.pi) % (2 * np.pi) - np.pi
    assert np.all(np.abs(bd - printed) <= 4e-3)
    assert np.all(np.abs(per_block[:-1, 9] - (borders[:, 4] - borders[:, 2])) <= 5e-3)
    # running total-count phase
    assert np.allclose(total, np.cumsum(blocks[:, 7]), atol=2e-2, rtol=0)


def _cubic_track(B, T, p):
    """Per-block Taylor coefficients of a globally cubic phase phi(t) = p0 + p1 t + p2 t^2 + p3 t^3."""
    tc = (np.arange(B) + 0.5) * T
    phi = p[0] + p[1] * tc + p[2] * tc**2 + p[3] * tc**3
    d1 = p[1] + 2 * p[2] * tc + 3 * p[3] * tc**2
    d2 = 2 * p[2] + 6 * p[3] * tc
    d3 = 6 * p[3] * np.ones(B)
    best = np.stack([np.ones(B), np.zeros(B), phi, d1 / (2 * np.pi), d2 / (2 * np.pi), d3 / (2 * np.pi)], axis=1)
    return best, lambda t: p[0] + p[1] * t + p[2] * t**2 + p[3] * t**3


def test_polynomial_phase_is_continuous_and_sums_to_the_analytic_integral():
    B, T = 120, 0.5
    p = [0.3, 2 * np.pi * 40.0, 2 * np.pi * 0.7, 2 * np.pi * 0.01]
    best, phi = _cubic_track(B, T, p)
    per_block, total, iv = oracle.doppler_products(best, T, blocks_per_interval=[2, 20, 120])
    assert np.all(np.abs(per_block[:-1, 8]) < 1e-8)          # border phase residuals vanish
    assert np.all(np.abs(per_block[:-1, 9]) < 1e-8)          # border frequency residuals vanish
    assert np.isnan(per_block[-1, 8]) and np.isnan(per_block[-1, 9])
    edges = np.arange(B + 1) * T
    assert np.allclose(per_block[:, 7], phi(edges[1:]) - phi(edges[:-1]), rtol=0, atol=1e-8)
    assert np.allclose(total, phi(edges[1:]) - phi(0.0), rtol=0, atol=1e-7)
    # Eq. 16-17: integration Doppler over Tc = m T
    for m, out in zip([2, 20, 120], iv):
        assert out.shape == (B // m, 2)
        e = np.arange(B // m + 1) * m * T
        assert np.allclose(out[:, 0], phi(e[1:]) - phi(e[:-1]), rtol=0, atol=1e-7)
        assert np.allclose(out[:, 1], out[:, 0] / (m * T), rtol=1e-15)
    # the long interval is the sum of the short ones
    assert abs(iv[2][0, 0] - iv[1][:, 0].sum()) < 1e-7
    assert abs(total[-1] - per_block[:, 7].sum()) < 1e-7


def test_invariants_frequency_is_the_phase_derivative():
    rng = np.random.default_rng(0)
    T = 1.0
    best = np.stack([np.ones(6), np.zeros(6), rng.uniform(-3, 3, 6), rng.uniform(100, 3000, 6),
                     rng.uniform(-5, 5, 6), rng.uniform(-1, 1, 6)], axis=1)
    pb, _, _ = oracle.doppler_products(best, T, los_scale=0.25)
    for k in range(6):
        f, fdot, fddot = best[k, 3], best[k, 4], best[k, 5]
        # F(+-T/2) = 2 pi (f +- fdot T/2 + fddot T^2/8); F(0) = 2 pi f is their mean minus the curvature term
        assert abs(pb[k, 6] - 2 * np.pi * (f + fdot * T / 2 + fddot * T * T / 8)) < 1e-9 * abs(pb[k, 6])
        assert abs(pb[k, 5] - 2 * np.pi * (f - fdot * T / 2 + fddot * T * T / 8)) < 1e-9 * abs(pb[k, 5])
        # Eq. 17 summand in closed form: 2 pi (f T + fddot T^3/24)
        assert abs(pb[k, 7] - 2 * np.pi * (f * T + fddot * T**3 / 24)) < 1e-9 * abs(pb[k, 7])
        # numerical derivative of the oracle's own model phase at +T/2 via the D=6 model at unit amplitude:
        h = 1e-6
        th = best[k].copy()
        # phase(t) recovered from the model through arccos is ill-conditioned; use the edge phases instead:
        # (phi(T/2) - phi(-T/2)) / T = mean frequency over the block = 2 pi (f + fddot T^2/24)
        assert abs(pb[k, 7] / T - 2 * np.pi * (f + fddot * T * T / 24)) < 1e-6
        assert pb[k, 0] == f and pb[k, 1] == fdot
        assert pb[k, 2] == 0.25 * fdot                          # Eq. 19: a_los = los_scale * fdot
        del h, th


def test_d5_has_no_cubic_term():
    best5 = np.array([[1.0, 0.0, 0.2, 100.0, 3.0]])
    best6 = np.array([[1.0, 0.0, 0.2, 100.0, 3.0, 0.0]])
    a, ta, _ = oracle.doppler_products(best5, 2.0)
    b, tb, _ = oracle.doppler_products(best6, 2.0)
    assert np.array_equal(a[:, :8], b[:, :8]) and np.array_equal(ta, tb)
    assert abs(a[0, 7] - 2 * np.pi * 100.0 * 2.0) < 1e-9


def test_border_wrap_is_in_minus_pi_pi():
    # two blocks whose border phases differ by almost a full turn: residual must come out small and signed
    T = 1.0
    b0 = [1, 0, 0.0, 10.0, 0.0]
    b1 = [1, 0, 0.05, 10.0, 0.0]       # phase at the border: left 0 + 2 pi 5 -> 0 ; right 0.05 - 2 pi 5 -> 0.05
    pb, _, _ = oracle.doppler_products(np.array([b0, b1], dtype=np.float64), T)
    assert abs(pb[0, 8] - 0.05) < 1e-9
    pb, _, _ = oracle.doppler_products(np.array([b1, b0], dtype=np.float64), T)
    assert abs(pb[0, 8] + 0.05) < 1e-9
    b2 = [1, 0, np.pi, 10.0, 0.0]
    pb, _, _ = oracle.doppler_products(np.array([b0, b2], dtype=np.float64), T)
    assert abs(abs(pb[0, 8]) - np.pi) < 1e-9
