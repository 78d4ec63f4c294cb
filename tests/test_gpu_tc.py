"""GPU parity of the tensor-core kernel (pt_tc_kernel: phase by tcgen05.mma kind::tf32 into TMEM) against the fp64 oracle, through
the C ABI.  PT_KERNEL=tc / classic is the library's documented test hook that forces one of the two evaluation kernels; the
automatic choice is exercised as well.  Bars are north_star's: fitness <= 1e-4 relative on identical populations, fitted
parameters |dphi0| < 5 mrad and |df| < 1e-3 Hz, bit-exact random streams (shared device functions: checked via trajectories)."""
import os

import numpy as np
import pytest

import oracle
from _observed import observed
from paper_1906_10598_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

FIT_REL_TOL, PHI0_TOL, F_TOL = 1e-4, 5e-3, 1e-3


@pytest.fixture(scope="module")
def pt():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device; there is no CPU fallback")
    from paper_1906_10598_b200 import pt as _pt
    _pt.lib()
    return _pt


class _kernel:
    def __init__(self, which):
        self.which = which

    def __enter__(self):
        self.old = {k: os.environ.get(k) for k in ("PT_KERNEL", "PT_CLUSTER")}
        os.environ["PT_KERNEL"] = self.which
        os.environ["PT_CLUSTER"] = "1"           # few-block inputs would otherwise take the cluster path of the classic kernel

    def __exit__(self, *a):
        for k, v in self.old.items():
            if v is None:
                os.environ.pop(k, None)
            else:
                os.environ[k] = v


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _wrap(d):
    return (np.asarray(d) + np.pi) % (2 * np.pi) - np.pi


def _fitness_both(pt, wl, NP, seed=0, spread=1.0, objective=0):
    rng = np.random.default_rng(seed)
    c = 0.5 * (wl.lo + wl.hi)
    h = 0.5 * (wl.hi - wl.lo) * spread
    pop = (c[:, None, :] + h[:, None, :] * rng.uniform(-1, 1, (wl.B, NP, wl.D))).astype(np.float32)
    if objective:
        pop[:, :, 1] = 0.0
    with _kernel("tc"):
        plan = pt.pt_fit_blocks_plan(wl.B, wl.N, pt.make_config(D=wl.D, NP=NP, generations=1, t0=wl.t0, objective=objective))
        assert plan["cands_per_thread"] == 1 and plan["threads"] == 640, plan       # the tensor-core plan
        got = pt.pt_objective(_cuda(wl.x), wl.fs, _cuda(pop), objective).cpu().numpy()
    ref = oracle.fitness(wl.x, wl.fs, pop, objective=objective)
    return got, ref, pop


@pytest.mark.parametrize("make,NP", [(lambda: W.config0(cases=range(5)), 60), (lambda: W.config1(blocks=[0, 59]), 100),
                                     (lambda: W.config2(blocks=[0, 1800, 3599]), 128), (lambda: W.config3(blocks=[0, 17950, 35999]), 128)])
def test_tc_fitness_parity_configs(pt, make, NP):
    wl = make()
    got, ref, _ = _fitness_both(pt, wl, NP, seed=NP)
    rel = np.abs(got - ref) / ref
    print("\n[tc fitness %s NP=%d] max rel err %.2e" % (wl.name, NP, rel.max()))
    assert rel.max() < FIT_REL_TOL
    got, ref, _ = _fitness_both(pt, wl, NP, seed=NP + 1, spread=1e-4)           # collapsed population
    assert np.max(np.abs(got - ref) / ref) < FIT_REL_TOL


@pytest.mark.parametrize("N,NP,D", [(8, 4, 5), (254, 5, 6), (256, 128, 5), (258, 33, 6), (1000, 97, 5), (4094, 128, 6), (40002, 64, 5)])
def test_tc_fitness_ragged_sizes(pt, N, NP, D):
    """Tiles of 256 samples with a ragged tail, fewer candidates than TMEM lanes, the smallest and the largest resident blocks."""
    rng = np.random.default_rng(N + NP)
    B, fs = 3, float(N)
    t = -0.5 + np.arange(N) / fs
    truth = np.array([1.0, 0.05, 0.3, 0.21 * N, 0.5, 0.2][:D])
    ph = truth[2] + 2 * np.pi * (truth[3] * t + truth[4] * t * t / 2 + (truth[5] * t**3 / 6 if D == 6 else 0.0))
    x = ((truth[0] + truth[1] * t) * np.cos(ph) + 0.1 * rng.standard_normal((B, N))).astype(np.float32)
    pop = (truth * (1 + 0.2 * rng.uniform(-1, 1, (B, NP, D)))).astype(np.float32)
    with _kernel("tc"):
        got = pt.pt_fitness(_cuda(x), fs, _cuda(pop)).cpu().numpy()
    ref = oracle.fitness(x, fs, pop)
    assert np.max(np.abs(got - ref) / ref) < FIT_REL_TOL


def test_tc_correlation_objective_parity(pt):
    """Eq. 5-6 through the tensor-core kernel, at the bars of tests/test_gpu_strategies_cor.py."""
    from test_gpu_strategies_cor import _objective_case
    wl = W.config2(blocks=[5, 2000])
    wl.lo = wl.lo.copy(); wl.hi = wl.hi.copy()
    wl.lo[:, 0] = wl.hi[:, 0] = wl.truth[:, 0]           # Eq. 6: constant, known amplitude
    wl.lo[:, 1] = wl.hi[:, 1] = 0.0
    with _kernel("tc"):
        e_cor, e_f = _objective_case(pt, wl, 128, seed=3)
        e_cor2, e_f2 = _objective_case(pt, wl, 128, seed=4, spread=1e-4)
    print("\n[tc cor] spread box: err_cor %.2e err_F %.2e; collapsed: %.2e %.2e" % (e_cor, e_f, e_cor2, e_f2))
    assert e_cor < 1e-4 and e_f < 1e-4 and e_cor2 < 1e-4 and e_f2 < 1e-4


def _fit(pt, wl, kernel, seed, want_pop=False, generations=None, strategy=1):
    de = wl.de
    cfg = pt.make_config(D=de["D"], NP=de["NP"], generations=de["generations"] if generations is None else generations, F=de["F"],
                         CR=de["CR"], seed=seed, t0=wl.t0, strategy=strategy)
    with _kernel(kernel):
        r = pt.pt_fit_blocks(_cuda(wl.x), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg, block_index=_cuda(wl.block_index.astype(np.int32)),
                             want_pop=want_pop)
        torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in r.items()}


def test_tc_first_generations_follow_the_oracle_trajectory(pt):
    """Generation 0 is bit-identical (same Philox words, same fp64 arithmetic); after a few generations almost every member still
    is (a selection decision can differ only where two objective values lie within the fp32 error)."""
    wl = W.config0(cases=range(6))
    for G in (0, 1, 5):
        g = _fit(pt, wl, "tc", seed=5, want_pop=True, generations=G)
        o = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=60, generations=G, seed=5, want_pop=True)
        same = np.all(g["final_pop"] == o["final_pop"].astype(np.float32), axis=-1)
        print("\n[tc trajectory] G=%d identical members %.4f" % (G, same.mean()))
        assert same.mean() == 1.0 if G == 0 else same.mean() > 0.98
        assert np.max(np.abs(g["final_fit"] - o["final_fit"]) / o["final_fit"]) < FIT_REL_TOL or G > 0


@pytest.mark.parametrize("make,seed", [(lambda: W.config0(cases=range(12)), 3), (lambda: W.config1(blocks=[0, 30]), 2),
                                       (lambda: W.config2(blocks=[0, 1800]), 2), (lambda: W.config3(blocks=[100, 30000]), 4)])
def test_tc_full_fit_vs_oracle(pt, make, seed):
    wl = make()
    g = _fit(pt, wl, "tc", seed=seed)
    de = wl.de
    o = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=de["NP"], generations=de["generations"], F=de["F"], CR=de["CR"], seed=seed,
                          block_index=wl.block_index)
    drss = np.abs(g["best_rss"] - o["best_rss"]) / o["best_rss"]
    same = drss < FIT_REL_TOL
    dphi, df = _wrap(g["best"][:, 2] - o["best"][:, 2]), g["best"][:, 3] - o["best"][:, 3]
    print("\n[tc fit %s] same optimum %d/%d, max |dphi0| %.2e rad, max |df| %.2e Hz, max dRSS %.2e" %
          (wl.name, same.sum(), wl.B, np.abs(dphi[same]).max(), np.abs(df[same]).max(), drss[same].max()))
    observed("identical members (bar >= 0.9)", round(float(same.mean()), 4))
    assert same.mean() >= 0.9
    assert np.abs(dphi[same]).max() < PHI0_TOL and np.abs(df[same]).max() < F_TOL
    for k in range(wl.B):           # every result is valid: its objective is the oracle's at its own parameters
        r = oracle.rss(wl.x[k], wl.fs, g["best"][k])
        assert abs(float(g["best_rss"][k]) - r) / r < FIT_REL_TOL
        assert np.all(g["best"][k] >= wl.lo[k]) and np.all(g["best"][k] <= wl.hi[k])


@pytest.mark.parametrize("strategy", [2, 3, 6])
def test_tc_strategies_agree_with_the_classic_kernel(pt, strategy):
    """The DE step is shared device code: with the same seed both kernels follow the same trajectory until a selection falls
    inside the fp32 error of the two (different) summation orders; both must land on the same optimum."""
    wl = W.config0(cases=range(8))
    a = _fit(pt, wl, "tc", seed=7, strategy=strategy, generations=300)
    b = _fit(pt, wl, "classic", seed=7, strategy=strategy, generations=300)
    same = np.abs(a["best_rss"] - b["best_rss"]) / b["best_rss"] < FIT_REL_TOL
    observed("identical members (bar >= 0.75)", round(float(same.mean()), 4))
    assert same.mean() >= 0.75
    assert np.abs(_wrap(a["best"][same, 2] - b["best"][same, 2])).max() < PHI0_TOL
    assert np.abs(a["best"][same, 3] - b["best"][same, 3]).max() < F_TOL


def test_tc_persistent_loop_block_index_quantised_and_status(pt):
    """More blocks than CTAs (every CTA loops), a sub-range reproduces the full launch bit for bit, quantised input equals fp32
    input on the unpacked samples, and the status bits (non-finite sample, inverted box) are set per block."""
    wl = W.single_tone_blocks(range(400), 512, 512.0, config=4, f_range=(20, 60))
    wl.de = dict(NP=32, D=5, generations=10, F=0.5, CR=0.9)
    x = wl.x.copy()
    x[77, 100] = np.nan
    lo = wl.lo.copy()
    lo[5, 3] = wl.hi[5, 3] + 1.0
    wl2 = W.single_tone_blocks(range(400), 512, 512.0, config=4, f_range=(20, 60))
    wl2.de, wl2.x, wl2.lo = wl.de, x, lo
    g = _fit(pt, wl2, "tc", seed=9, want_pop=True)
    assert list(np.nonzero(g["status"] & 8)[0]) == [77] and list(np.nonzero(g["status"] & 16)[0]) == [5]
    sub = W.single_tone_blocks([300], 512, 512.0, config=4, f_range=(20, 60))
    sub.de = wl.de
    sub.block_index = np.array([300], dtype=np.uint32)
    gs = _fit(pt, sub, "tc", seed=9, want_pop=True)
    assert np.array_equal(gs["final_pop"][0], g["final_pop"][300]) and np.array_equal(gs["best"][0], g["best"][300])
    xq, qd = W.quantise(wl.x[:40], 8)
    quant = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
    cfg = pt.make_config(D=5, NP=32, generations=10, seed=9, t0=wl.t0)
    with _kernel("tc"):
        xf = pt.pt_unpack_samples(_cuda(xq), 512, quant)
        a = pt.pt_fit_blocks(_cuda(xq), wl.fs, _cuda(wl.lo[:40]), _cuda(wl.hi[:40]), cfg, quant=quant, N=512)
        b = pt.pt_fit_blocks(xf, wl.fs, _cuda(wl.lo[:40]), _cuda(wl.hi[:40]), cfg)
        torch.cuda.synchronize()
    assert torch.equal(a["best"], b["best"]) and torch.equal(a["best_rss"], b["best_rss"])


def test_automatic_choice_is_the_run_kernel_and_the_hooks_force_the_others(pt):
    """Automatic choice: pt_run_kernel everywhere -- 1024 threads per SM as 1, 2 or 4 CTAs, one candidate per
    thread; PT_KERNEL=tc / classic force the other two evaluation kernels."""
    cfg6 = pt.make_config(D=6, NP=128, generations=1500, t0=-0.05)
    cfg5 = pt.make_config(D=5, NP=128, generations=1000, t0=-0.5)
    for B, N, cfg in ((36000, 10000, cfg6), (3600, 16000, cfg5), (1024, 4096, cfg5), (1024, 262144, cfg5)):
        plan = pt.pt_fit_blocks_plan(B, N, cfg)
        assert plan["threads"] * plan["ctas_per_sm"] == 1024 and plan["cands_per_thread"] == 1, plan
    with _kernel("tc"):
        assert pt.pt_fit_blocks_plan(36000, 10000, cfg6)["threads"] == 640
    with _kernel("classic"):
        assert pt.pt_fit_blocks_plan(3600, 16000, cfg5)["threads"] == 512


def test_classic_kernel_still_covers_d6(pt):
    """The automatic choice is pt_run_kernel; the D = 6 paths of the other two kernels stay covered: both on
    the same config-3 blocks against the oracle's objective, and against each other at the parity bars."""
    wl = W.config3(blocks=[100, 20000])
    a = _fit(pt, wl, "classic", seed=4)
    b = _fit(pt, wl, "tc", seed=4)
    for r in (a, b):
        for k in range(wl.B):
            v = oracle.rss(wl.x[k], wl.fs, r["best"][k])
            assert abs(float(r["best_rss"][k]) - v) / v < FIT_REL_TOL
    assert np.abs(_wrap(a["best"][:, 2] - b["best"][:, 2])).max() < PHI0_TOL
    assert np.abs(a["best"][:, 3] - b["best"][:, 3]).max() < F_TOL


def test_tc_main_launch_with_classic_cluster_tail(pt):
    """B = 2 waves + a short tail: full waves on the tensor-core kernel (two blocks per CTA), the tail on clusters of the FP32-pipe
    kernel (two launches).  Every block must equal its single-block fit up to the summation order of its kernel."""
    wl = W.single_tone_blocks(range(310), 512, 512.0, config=4, f_range=(20, 60))
    wl.de = dict(NP=16, D=5, generations=6, F=0.5, CR=0.9)
    cfg = pt.make_config(D=5, NP=16, generations=6, seed=9, t0=wl.t0)
    old = os.environ.get("PT_KERNEL")
    os.environ["PT_KERNEL"] = "tc"
    try:
        plan = pt.pt_fit_blocks_plan(wl.B, wl.N, cfg)
        assert plan["threads"] == 640 and plan["tail_cluster"] >= 2, plan
        r = pt.pt_fit_blocks(_cuda(wl.x), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg, want_pop=True)
        torch.cuda.synchronize()
    finally:
        if old is None:
            os.environ.pop("PT_KERNEL", None)
        else:
            os.environ["PT_KERNEL"] = old
    g = {k: v.cpu().numpy() for k, v in r.items()}
    assert np.all(np.isfinite(g["best_rss"])) and np.all(g["best"] >= wl.lo) and np.all(g["best"] <= wl.hi)
    o = oracle.fit_blocks(wl.x[[0, 200, 305]], wl.fs, wl.lo[[0, 200, 305]], wl.hi[[0, 200, 305]], NP=16, generations=6, seed=9,
                          block_index=np.array([0, 200, 305], dtype=np.uint32), want_pop=True)
    same = np.all(g["final_pop"][[0, 200, 305]] == o["final_pop"].astype(np.float32), axis=-1)
    observed("identical members (bar > 0.9)", round(float(same.mean()), 4))
    assert same.mean() > 0.9
