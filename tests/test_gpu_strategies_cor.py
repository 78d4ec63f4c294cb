"""GPU parity of the widened rows: f-3, the six mutation strategies of Table 4 (
DESIGN.md reading R21), and f-2, the correlation objective of Eq. 5-6 (reading R22) -- the CUDA path
through the C ABI against the fp64 oracle on the same seeded inputs.

Bars: trial vectors are fp64 without contraction on both sides, so populations are identical until a selection falls
inside the fp32 objective error; fitted phi0 within 5 mrad and f within 1e-3 Hz of the oracle's; objective values
within 1e-4 relative (for Eq. 5 on the correlation sum and on F_cor - 1/pi, the value the library reports).
"""
import numpy as np
import pytest

import oracle
from _observed import observed
from paper_1906_10598_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

REL_TOL = 1e-4
PHI0_TOL = 5e-3
F_TOL = 1e-3


@pytest.fixture(scope="module")
def pt():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device; there is no CPU fallback")
    from paper_1906_10598_b200 import pt as _pt
    _pt.lib()
    return _pt


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _wrap(d):
    return (np.asarray(d) + np.pi) % (2 * np.pi) - np.pi


class _forced_cluster:
    def __init__(self, K):
        self.K = K

    def __enter__(self):
        import os
        self.old = os.environ.get("PT_CLUSTER")
        os.environ["PT_CLUSTER"] = str(self.K)

    def __exit__(self, *a):
        import os
        if self.old is None:
            os.environ.pop("PT_CLUSTER", None)
        else:
            os.environ["PT_CLUSTER"] = self.old


def _both(pt, wl, lo, hi, *, NP, G, F, CR, seed, strategy, objective=0, D=None):
    D = D or wl.D
    cfg = pt.make_config(D=D, NP=NP, generations=G, F=F, CR=CR, seed=seed, t0=wl.t0, strategy=strategy, objective=objective)
    r = pt.pt_fit_blocks(_cuda(wl.x), wl.fs, _cuda(lo), _cuda(hi), cfg, block_index=_cuda(wl.block_index.astype(np.int32)),
                         want_pop=True)
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in r.items()}
    o = oracle.fit_blocks(wl.x, wl.fs, lo, hi, NP=NP, generations=G, F=F, CR=CR, seed=seed, block_index=wl.block_index,
                          want_pop=True, strategy=strategy, objective=objective)
    return g, o


# ----------------------------------------------------------------------------------------------
# f-3: mutation strategies
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("strategy", [2, 3, 4, 5, 6])
@pytest.mark.parametrize("D", [5, 6])
def test_first_generations_follow_the_oracle_trajectory(pt, strategy, D):
    wl = W.config0(cases=range(4)) if D == 5 else W.config3(blocks=[17990, 18010], NP=60, generations=5)
    for G, F, CR in ((1, 0.5, 0.9), (4, 1.7, 0.6)):
        g, o = _both(pt, wl, wl.lo, wl.hi, NP=60, G=G, F=F, CR=CR, seed=31 + strategy, strategy=strategy)
        same = np.all(g["final_pop"] == o["final_pop"].astype(np.float32), axis=-1)
        # config 3 (T = 0.1 s) does not observe fdot, fddot, a1 (R13): trials that differ only there have RSS values
        # inside the fp32 error, so more selections flip, and a flipped member spreads through the difference vectors
        floor = 0.97 if (D == 5 or G == 1) else 0.8
        observed("identical members (bar > floor)", round(float(same.mean()), 4))
        assert same.mean() > floor, (strategy, G, same.mean())
        assert np.max(np.abs(g["final_fit"] - o["final_fit"])[same] / o["final_fit"][same]) < REL_TOL
        assert np.all(g["final_pop"] >= wl.lo[:, None, :].astype(np.float32) - 1e-6)
        assert np.all(g["final_pop"] <= wl.hi[:, None, :].astype(np.float32) + 1e-6)


@pytest.mark.parametrize("strategy", [2, 3])
def test_best_guided_strategies_on_clusters(pt, strategy):
    """The best member is found redundantly by every CTA of a cluster from bit-identical RSS values."""
    wl = W.config0(cases=range(3))
    with _forced_cluster(4):
        g, o = _both(pt, wl, wl.lo, wl.hi, NP=64, G=3, F=0.6, CR=0.9, seed=7, strategy=strategy)
    same = np.all(g["final_pop"] == o["final_pop"].astype(np.float32), axis=-1)
    observed("identical members (bar > 0.97)", round(float(same.mean()), 4))
    assert same.mean() > 0.97


@pytest.mark.parametrize("strategy,F,CR,G", [(2, 0.5, 0.9, 400), (3, 0.7, 0.9, 400), (4, 0.5, 0.9, 500), (5, 0.3, 0.9, 500),
                                             (6, 0.5, 0.9, 500)])
def test_full_fits_agree_with_the_oracle(pt, strategy, F, CR, G):
    """DE is a heuristic (R19): after the first selection that falls inside the fp32 / fp64 difference of the objective the two
    trajectories are different random searches, and the best-guided strategies stall on some blocks on either side.  What is
    asserted: nothing beats the global optimum (a DE/rand/1 fit of 500 generations by the oracle); the GPU reaches it on about as
    many blocks as the oracle does (the two fractions are printed); where both reached it the parameters agree at the parity
    bars; every GPU result is valid."""
    wl = W.config0(cases=range(8))
    g, o = _both(pt, wl, wl.lo, wl.hi, NP=60, G=G, F=F, CR=CR, seed=13, strategy=strategy)
    ref = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=500, F=0.5, CR=0.9, seed=13)
    at_g = np.abs(g["best_rss"] - ref["best_rss"]) <= 1e-5 * ref["best_rss"]
    at_o = np.abs(o["best_rss"] - ref["best_rss"]) <= 1e-5 * ref["best_rss"]
    print("\n[strategy %d] blocks at the global optimum: GPU %d / 8, oracle %d / 8, both %d" % (strategy, at_g.sum(), at_o.sum(), (at_g & at_o).sum()))
    for res in (g, o):
        assert np.all(res["best_rss"] >= ref["best_rss"] * (1 - 1e-5))
    assert at_g.sum() >= at_o.sum() - 2 and at_g.sum() >= 4
    ok = at_g & at_o
    assert np.max(np.abs(_wrap(g["best"][ok, 2] - o["best"][ok, 2]))) < PHI0_TOL
    assert np.max(np.abs(g["best"][ok, 3] - o["best"][ok, 3])) < F_TOL
    # every result is valid: the reported RSS is the oracle's objective at the GPU's own parameters
    for k in range(wl.B):
        assert abs(g["best_rss"][k] - oracle.rss(wl.x[k], wl.fs, g["best"][k])) < REL_TOL * g["best_rss"][k]


def test_table4_settings_with_the_papers_strategy(pt):
    """Table 4: strategy 3, F_XC = 0.5, CR_XC = 0.85, itermax = 200.  best/1 converges fast and may
    stall (the paper re-searches such blocks): parameters are compared where both sides reached the same
    optimum; every result must be valid; most blocks converge."""
    wl = W.config0(cases=range(16))
    g, o = _both(pt, wl, wl.lo, wl.hi, NP=60, G=200, F=0.5, CR=0.85, seed=4, strategy=3)
    ref = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=500, F=0.5, CR=0.9, seed=4)
    ok = np.abs(g["best_rss"] - o["best_rss"]) <= 1e-5 * o["best_rss"]
    observed("fraction on the same optimum (bar >= 0.5)", ok.mean())
    assert ok.mean() >= 0.5
    assert np.max(np.abs(_wrap(g["best"][ok, 2] - o["best"][ok, 2]))) < PHI0_TOL
    assert np.max(np.abs(g["best"][ok, 3] - o["best"][ok, 3])) < F_TOL
    for res in (g, o):
        assert np.all(res["best_rss"] >= ref["best_rss"] * (1 - 1e-5))          # nothing beats the global optimum
        assert np.mean(res["best_rss"] <= ref["best_rss"] * 1.01) >= 0.75       # and most blocks are within 1 % of it
    for k in range(wl.B):
        assert abs(g["best_rss"][k] - oracle.rss(wl.x[k], wl.fs, g["best"][k])) < REL_TOL * g["best_rss"][k]


def test_invalid_strategy_and_objective_are_rejected(pt):
    wl = W.config0(cases=[0])
    for kw in (dict(strategy=7), dict(strategy=-1), dict(objective=2)):
        cfg = pt.make_config(D=5, NP=16, generations=1, t0=wl.t0, **kw)
        with pytest.raises(pt.PtError):
            pt.pt_fit_blocks(_cuda(wl.x), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg)
    # strategy 0 (a zero-initialised record) is DE/rand/1
    a = pt.pt_fit_blocks(_cuda(wl.x), wl.fs, _cuda(wl.lo), _cuda(wl.hi),
                         pt.make_config(D=5, NP=16, generations=3, t0=wl.t0, strategy=0), want_pop=True)
    b = pt.pt_fit_blocks(_cuda(wl.x), wl.fs, _cuda(wl.lo), _cuda(wl.hi),
                         pt.make_config(D=5, NP=16, generations=3, t0=wl.t0, strategy=1), want_pop=True)
    assert torch.equal(a["final_pop"], b["final_pop"])


# ----------------------------------------------------------------------------------------------
# f-2: correlation objective
# ----------------------------------------------------------------------------------------------
def _cor_of_reported(fm):
    """Invert the reported value F_cor - 1/pi (fp64): cor = tan(1/F_cor - pi/2)."""
    g = 1.0 / (np.asarray(fm, dtype=np.float64) + 1.0 / np.pi)          # arctan(cor) + pi/2
    return -1.0 / np.tan(g)                                             # tan(g - pi/2) = -cot(g)


def _objective_case(pt, wl, NP, seed=0, spread=1.0):
    rng = np.random.default_rng(seed)
    D = wl.D
    mid, half = 0.5 * (wl.lo + wl.hi), 0.5 * (wl.hi - wl.lo) * spread
    pop = (mid[:, None, :] + half[:, None, :] * rng.uniform(-1, 1, size=(wl.B, NP, D))).astype(np.float32)
    ref = oracle.fitness(wl.x, wl.fs, pop, objective=1)                 # F_cor, fp64
    got = pt.pt_objective(_cuda(wl.x), wl.fs, _cuda(pop), 1).cpu().numpy().astype(np.float64)
    ref_cor = _cor_of_reported(ref - 1.0 / np.pi)
    got_cor = _cor_of_reported(got)
    # Tolerance.  A correlation sum of a far-off candidate is a sum of N terms of either sign that nearly
    # cancel, so its error is not relative to |cor| but to the terms: the fp32 phase argument carries 2^-24 of the
    # candidate's offset from the block's reference (up to ~1e3 rad in a +-20 % box -> ~1e-4 rad per sample, random in
    # sign), which moves the sum by ~1e-4 sqrt(N) rms(x) a0.  Bar: 1e-4 |cor| + 1e-5 a0 sqrt(sum x^2 N/2) (the second term
    # is 1e-5 of the largest correlation Cauchy-Schwarz allows).  Where the candidate correlates (|cor| > 10 % of that
    # scale) the reported F_cor - 1/pi itself is held to 1e-4 relative.
    scale = np.abs(pop[..., 0].astype(np.float64)) * np.sqrt(np.sum(wl.x.astype(np.float64) ** 2, axis=1) * wl.N / 2)[:, None]
    err_cor = np.abs(got_cor - ref_cor) / (np.abs(ref_cor) + 0.1 * scale)
    big = np.abs(ref_cor) > 0.1 * scale
    err_f = np.abs(got - (ref - 1.0 / np.pi))[big] / (ref - 1.0 / np.pi)[big]
    return err_cor.max(), (err_f.max() if big.any() else 0.0)


def test_objective_cor_on_given_populations(pt):
    for wl, NP in ((W.config0(cases=range(6), a1_zero=True), 60), (W.config2(blocks=[0, 1799, 3599]), 128),
                   (W.config3(blocks=[0, 18000, 35999]), 128), (W.config1(blocks=[0, 59]), 100)):
        e_cor, e_f = _objective_case(pt, wl, NP)
        assert e_cor < REL_TOL and e_f < REL_TOL, (wl.name, e_cor, e_f)
        # collapsed population: |cor| ~ a0 A N/2, both measures far below the bar
        e_cor, e_f = _objective_case(pt, wl, NP, spread=1e-4)
        assert e_cor < 1e-5 and e_f < 1e-5, (wl.name, e_cor, e_f)


@pytest.mark.parametrize("N,NP", [(8, 4), (130, 7), (1030, 13), (16384, 512)])
def test_objective_cor_ragged_sizes(pt, N, NP):
    wl = W.single_tone_blocks(range(4), N, float(N), config=4, f_range=(0.05 * N, 0.2 * N), a1_zero=True)
    e_cor, e_f = _objective_case(pt, wl, NP, seed=N)
    assert e_cor < REL_TOL and e_f < REL_TOL


def test_objective_cor_streamed_and_chi2_entry_unchanged(pt):
    with _forced_cluster(1):
        wl = W.single_tone_blocks(range(2), 65536 + 132, 65536.0, config=4, f_range=(50.0, 200.0), a1_zero=True)
        e_cor, e_f = _objective_case(pt, wl, 24, seed=5)
        assert e_cor < REL_TOL and e_f < REL_TOL
    wl = W.config0(cases=range(2))
    pop = np.repeat(wl.truth[:, None, :], 8, axis=1).astype(np.float32)
    a = pt.pt_objective(_cuda(wl.x), wl.fs, _cuda(pop), 0)
    b = pt.pt_fitness(_cuda(wl.x), wl.fs, _cuda(pop))
    assert torch.equal(a, b)


def _cor_box(wl):
    lo, hi = wl.lo.copy(), wl.hi.copy()
    lo[:, 0] = hi[:, 0] = wl.truth[:, 0]           # Eq. 6: constant amplitude, "the average amplitude of signal"
    lo[:, 1] = hi[:, 1] = 0.0
    return lo, hi


@pytest.mark.parametrize("strategy", [6, 1])
def test_cor_fit_config0(pt, strategy):
    """Strategy 6 is the paper's choice for Eq. 5."""
    wl = W.config0(cases=range(8), a1_zero=True)
    lo, hi = _cor_box(wl)
    # generation 0 and the first generations: identical populations
    g, o = _both(pt, wl, lo, hi, NP=60, G=3, F=0.5, CR=0.9, seed=2, strategy=strategy, objective=1)
    same = np.all(g["final_pop"] == o["final_pop"].astype(np.float32), axis=-1)
    observed("identical members (bar > 0.97)", round(float(same.mean()), 4))
    assert same.mean() > 0.97
    g, o = _both(pt, wl, lo, hi, NP=60, G=400, F=0.5, CR=0.9, seed=2, strategy=strategy, objective=1)
    assert np.max(np.abs(_wrap(g["best"][:, 2] - o["best"][:, 2]))) < PHI0_TOL
    assert np.max(np.abs(g["best"][:, 3] - o["best"][:, 3])) < F_TOL
    fm_o = o["best_rss"] - 1.0 / np.pi
    assert np.max(np.abs(g["best_rss"] - fm_o) / fm_o) < REL_TOL
    assert np.max(np.abs(g["final_fit"] - (o["final_fit"] - 1.0 / np.pi)) / (o["final_fit"] - 1.0 / np.pi)) < REL_TOL
    assert np.all(g["status"] == o["status"]) and np.all((g["status"] & 2) == 0)
    # versus the generating truth: the maximiser of the correlation is the least-squares phase up to the noise
    assert np.max(np.abs(_wrap(g["best"][:, 2] - wl.truth[:, 2]))) < 0.05
    assert np.max(np.abs(g["best"][:, 3] - wl.truth[:, 3])) < 0.02


def test_cor_fit_config2_blocks_and_clusters(pt):
    """Config 2 blocks (N = 16000, NP = 128, 0 dB) under Eq. 5 with the sixth strategy; the same blocks split over
    clusters of 4 CTAs give the same populations up to the fp32 summation order."""
    wl = W.config2(blocks=[0, 900, 1800, 3599])
    lo, hi = wl.lo.copy(), wl.hi.copy()
    lo[:, 0] = hi[:, 0] = 1.0
    lo[:, 1] = hi[:, 1] = 0.0
    with _forced_cluster(1):
        g, o = _both(pt, wl, lo, hi, NP=128, G=300, F=0.5, CR=0.9, seed=6, strategy=6, objective=1)
    assert np.max(np.abs(_wrap(g["best"][:, 2] - o["best"][:, 2]))) < PHI0_TOL
    assert np.max(np.abs(g["best"][:, 3] - o["best"][:, 3])) < F_TOL
    fm_o = o["best_rss"] - 1.0 / np.pi
    assert np.max(np.abs(g["best_rss"] - fm_o) / fm_o) < REL_TOL
    with _forced_cluster(4):
        g4, _ = _both(pt, wl, lo, hi, NP=128, G=300, F=0.5, CR=0.9, seed=6, strategy=6, objective=1)
    assert np.max(np.abs(_wrap(g4["best"][:, 2] - g["best"][:, 2]))) < PHI0_TOL
    assert np.max(np.abs(g4["best"][:, 3] - g["best"][:, 3])) < F_TOL
    assert np.max(np.abs(g4["best_rss"] - g["best_rss"]) / g["best_rss"]) < REL_TOL


def test_cor_diverges_with_a_free_amplitude(pt):
    """"otherwise, the objective function becomes divergent" -- a0 runs to its upper bound on both sides."""
    wl = W.config0(cases=range(2), a1_zero=True)
    g, o = _both(pt, wl, wl.lo, wl.hi, NP=40, G=200, F=0.5, CR=0.9, seed=5, strategy=1, objective=1)
    for res in (g, o):
        assert np.all(np.abs(res["best"][:, 0] - wl.hi[:, 0]) <= 1e-3 * (wl.hi[:, 0] - wl.lo[:, 0]))


# ----------------------------------------------------------------------------------------------
# constant amplitude under the chi^2 objective: a1 fixed at zero takes the shorter evaluation loop
# ----------------------------------------------------------------------------------------------
def test_fixed_zero_amplitude_slope(pt):
    """The caller's a1 box is [0, 0]: the kernel drops the amplitude FFMA2 (a per-block run-time choice).  Objective values
    and fits against the oracle, resident / streamed / cluster paths, and blocks with and without the fixed slope mixed in
    one launch."""
    wl = W.config0(cases=range(6), a1_zero=True)
    lo, hi = wl.lo.copy(), wl.hi.copy()
    lo[:, 1] = hi[:, 1] = 0.0
    lo[3:, 1], hi[3:, 1] = -0.05, 0.05                           # blocks 3..5 keep a free slope
    rng = np.random.default_rng(0)
    pop = (lo[:, None, :] + (hi - lo)[:, None, :] * rng.uniform(0, 1, size=(6, 64, 5))).astype(np.float32)
    ref = oracle.fitness(wl.x, wl.fs, pop)
    got = pt.pt_fitness(_cuda(wl.x), wl.fs, _cuda(pop)).cpu().numpy()
    assert np.all(pop[:3, :, 1] == 0) and np.any(pop[3:, :, 1] != 0)
    assert np.max(np.abs(got - ref) / ref) < REL_TOL
    for K in (1, 4):
        with _forced_cluster(K):
            g, o = _both(pt, wl, lo, hi, NP=60, G=400, F=0.5, CR=0.9, seed=12, strategy=1)
        assert np.all(g["best"][:3, 1] == 0.0)
        assert np.max(np.abs(_wrap(g["best"][:, 2] - o["best"][:, 2]))) < PHI0_TOL
        assert np.max(np.abs(g["best"][:, 3] - o["best"][:, 3])) < F_TOL
        assert np.max(np.abs(g["best_rss"] - o["best_rss"]) / o["best_rss"]) < REL_TOL
    # streamed blocks, ragged tail
    with _forced_cluster(1):
        ws = W.single_tone_blocks(range(2), 65536 + 132, 65536.0, config=4, f_range=(50.0, 200.0), a1_zero=True)
        pop = np.repeat(ws.truth[:, None, :], 16, axis=1)
        pop[:, :, 3] += np.linspace(-0.2, 0.2, 16)[None, :]
        pop = pop.astype(np.float32)
        assert np.all(pop[:, :, 1] == 0)
        ref = oracle.fitness(ws.x, ws.fs, pop)
        got = pt.pt_fitness(_cuda(ws.x), ws.fs, _cuda(pop)).cpu().numpy()
        assert np.max(np.abs(got - ref) / ref) < REL_TOL
