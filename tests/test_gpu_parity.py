"""GPU parity tests: the CUDA path (through the C ABI, via the ctypes binding) against the fp64 CPU oracle,
element by element on the same seeded inputs.  Bars (BASELINE.json north_star / SURVEY.md 8(c)-(d)):
  * RNG streams and trial-vector indices: bit-exact;
  * generation-0 population: bit-exact in fp64;
  * fitness on identical populations: <= 1e-4 relative (fp32 + hardware cosine vs fp64);
  * fitted parameters vs the oracle on the same noisy block: |dphi0| < 5 mrad (wrapped), |df| < 1e-3 Hz;
  * both vs the generating truth: within 4 Cramer-Rao sigma;
  * Doppler products: <= 1e-9 relative on identical parameters.
"""
import numpy as np
import pytest

import oracle
from _observed import observed
from paper_1906_10598_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

FIT_REL_TOL = 1e-4      # north_star: "GPU fitness values must match the oracle within 1e-4 relative"
PHI0_TOL = 5e-3         # rad
F_TOL = 1e-3            # Hz


@pytest.fixture(scope="module")
def pt():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device; there is no CPU fallback")
    from paper_1906_10598_b200 import pt as _pt
    _pt.lib()
    return _pt


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class _forced_cluster:
    """PT_CLUSTER=<K> overrides the library's automatic cluster size (include/pt.h, pt_fit_blocks_plan)."""

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


@pytest.fixture
def no_cluster():
    """Few blocks would otherwise be split over a thread-block cluster (and large blocks become resident that way);
    the streamed-path tests pin the single-CTA plan."""
    with _forced_cluster(1):
        yield


def _wrap(d):
    return (np.asarray(d) + np.pi) % (2 * np.pi) - np.pi


def _crlb(theta, N, fs, sigma, D):
    """Cramer-Rao 1-sigma bounds of the model's parameters in white noise (Fisher matrix of Eq. 2)."""
    t = -N / (2 * fs) + np.arange(N) / fs
    th = list(theta) + [0.0] * (6 - len(theta))
    ph = th[2] + 2 * np.pi * (th[3] * t + th[4] * t * t / 2 + th[5] * t**3 / 6)
    A = th[0] + th[1] * t
    c, s = np.cos(ph), np.sin(ph)
    J = [c, t * c, -A * s, -A * s * 2 * np.pi * t, -A * s * np.pi * t * t]
    if D == 6:
        J.append(-A * s * np.pi * t**3 / 3)
    J = np.array(J)
    cov = np.linalg.inv(J @ J.T / sigma**2)
    return np.sqrt(np.diag(cov))


# ----------------------------------------------------------------------------------------------
# bit-exact integer work
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("NP,D,CR", [(4, 5, 0.9), (5, 6, 0.5), (60, 5, 0.9), (100, 5, 0.85), (128, 6, 0.9),
                                     (512, 5, 1.0), (1024, 6, 0.0)])
def test_de_draws_bit_exact(pt, NP, D, CR):
    rng = np.random.default_rng(NP * 10 + D)
    Q = 3000
    q = np.stack([rng.integers(0, 40000, Q), rng.integers(1, 2000, Q), rng.integers(0, NP, Q)], axis=1).astype(np.int32)
    q[:NP, 2] = np.arange(NP)                   # every candidate index at least once
    q[0, 0] = 2**31 - 1                         # large block index
    seed = 0xC0FFEE1234567 + NP
    got = pt.pt_de_draws(_cuda(q), NP, D, CR, seed).cpu().numpy()
    for k in range(Q):
        exp = oracle.de_draws(seed, int(q[k, 0]), int(q[k, 1]), int(q[k, 2]), NP, D, CR)
        assert tuple(int(v) for v in got[k]) == exp, (k, q[k])


@pytest.mark.parametrize("D", [5, 6])
def test_initial_population_bit_exact(pt, D):
    rng = np.random.default_rng(D)
    B, NP = 7, 33
    lo = rng.uniform(-5, 5, (B, D))
    hi = lo + rng.uniform(0, 3, (B, D))
    hi[2, 1] = lo[2, 1]                          # zero-width coordinate
    bidx = np.array([0, 1, 5, 77, 3599, 35999, 2**31 - 1], dtype=np.int32)
    seed = 987654321987
    got = pt.pt_init_population(_cuda(lo), _cuda(hi), NP, seed, _cuda(bidx)).cpu().numpy()
    for b in range(B):
        for i in range(NP):
            u = oracle.init_uniforms(seed, int(bidx[b]), i, D)
            assert np.array_equal(got[b, i], lo[b] + (hi[b] - lo[b]) * u)


# ----------------------------------------------------------------------------------------------
# fitness on identical populations
# ----------------------------------------------------------------------------------------------
def _fitness_case(pt, wl, NP, seed=0, spread=1.0):
    rng = np.random.default_rng(seed)
    D = wl.D
    mid, half = 0.5 * (wl.lo + wl.hi), 0.5 * (wl.hi - wl.lo) * spread
    pop = (mid[:, None, :] + half[:, None, :] * rng.uniform(-1, 1, size=(wl.B, NP, D))).astype(np.float32)
    ref = oracle.fitness(wl.x, wl.fs, pop)
    got = pt.pt_fitness(_cuda(wl.x), wl.fs, _cuda(pop)).cpu().numpy().astype(np.float64)
    rel = np.abs(got - ref) / ref
    return rel.max()


def test_fitness_config0(pt):
    assert _fitness_case(pt, W.config0(cases=range(6)), NP=60) < FIT_REL_TOL            # C = 4 path, ragged tail chunk
    assert _fitness_case(pt, W.config0(cases=range(3), box="paper"), NP=64) < FIT_REL_TOL


def test_fitness_config1_2_3(pt):
    assert _fitness_case(pt, W.config1(blocks=[0, 30, 59]), NP=100) < FIT_REL_TOL       # N = 10000: 78 chunks + 16 samples
    assert _fitness_case(pt, W.config2(blocks=[0, 1799, 3599]), NP=128) < FIT_REL_TOL   # C = 8 path, N = 16000
    assert _fitness_case(pt, W.config3(blocks=[0, 17900, 18000, 35999]), NP=128) < FIT_REL_TOL   # D = 6
    assert _fitness_case(pt, W.config3(blocks=[17000, 18100], box="paper"), NP=36) < FIT_REL_TOL


@pytest.mark.parametrize("N,NP", [(8, 4), (130, 7), (1030, 13), (4096, 32), (16384, 512), (2048, 1024)])
def test_fitness_ragged_sizes(pt, N, NP):
    """Smallest sizes, N not a multiple of the 128-sample chunk, NP not a multiple of the register blocking."""
    fs = float(N)
    wl = W.single_tone_blocks(range(5), N, fs, config=4, f_range=(0.05 * N, 0.2 * N))
    assert _fitness_case(pt, wl, NP=NP, seed=N) < FIT_REL_TOL


def test_fitness_near_converged_population_is_much_tighter(pt):
    """With the population collapsed around the optimum the offsets from the fp64 reference are tiny and the
    fp32 evaluation agrees with fp64 far better than the bar."""
    wl = W.config2(blocks=[10, 2000])
    assert _fitness_case(pt, wl, NP=128, spread=1e-4) < 2e-6


def test_fitness_unaligned_rows_take_the_non_bulk_path(pt):
    wl = W.single_tone_blocks(range(3), 1002, 1002.0, config=4, f_range=(50, 200))     # N % 4 == 2
    assert _fitness_case(pt, wl, NP=16) < FIT_REL_TOL


# ----------------------------------------------------------------------------------------------
# streamed path: blocks larger than shared memory (BASELINE config 4: 64 K and 256 K samples)
# ----------------------------------------------------------------------------------------------
class _forced_kernel:
    """PT_KERNEL=run / classic / tc forces one of the evaluation kernels (include/pt.h); unset = the automatic choice."""

    def __init__(self, which):
        self.which = which

    def __enter__(self):
        import os
        self.old = os.environ.get("PT_KERNEL")
        if self.which:
            os.environ["PT_KERNEL"] = self.which

    def __exit__(self, *a):
        import os
        if self.old is None:
            os.environ.pop("PT_KERNEL", None)
        else:
            os.environ["PT_KERNEL"] = self.old


@pytest.mark.parametrize("kernel,N,NP,B", [
    ("", 65536, 32, 3), ("", 65536, 512, 2), ("", 262144, 64, 2), ("", 65536 + 130, 40, 2), ("", 65536 + 132, 24, 2), ("", 70002, 16, 2),
    ("", 60000, 12, 150), ("", 65536, 1024, 1), ("", 100000 + 2, 400, 1),
    ("classic", 65536, 32, 3), ("classic", 65536 + 130, 40, 2), ("classic", 70002, 16, 2), ("classic", 30000, 12, 150),
    ("classic", 32768, 1024, 1)])
def test_fitness_streamed_blocks(pt, no_cluster, kernel, N, NP, B):
    """Tiles of the block move through the shared-memory ring; partial last tile, partial last run / chunk, rows that are
    not 16-byte aligned (N % 4 == 2: copied to the workspace first), more blocks than CTAs, more members than threads; both
    kernels that have a streamed path (the automatic pt_run_kernel and pt_block_kernel)."""
    with _forced_kernel(kernel):
        cfg = pt.make_config(D=5, NP=NP, generations=1, t0=0.0)
        assert pt.pt_fit_blocks_plan(B, N, cfg)["resident"] == 0
        wl = W.single_tone_blocks(range(B), N, float(N), config=4, f_range=(50.0, 200.0))
        assert _fitness_case(pt, wl, NP=NP, seed=N + NP) < FIT_REL_TOL


def test_fit_streamed_trajectory_and_full_fit(pt, no_cluster):
    """Config 4 point N = 65536, NP = 32, 200 generations on 4 blocks: first generations reproduce the oracle's
    population member by member; the full fit lands on the oracle's optimum."""
    wl = W.config4(65536, 32, B=4)
    assert pt.pt_fit_blocks_plan(wl.B, wl.N, pt.make_config(D=5, NP=32, generations=200, t0=wl.t0))["resident"] == 0
    g = _gpu_fit(pt, wl, generations=3, seed=4, want_pop=True)
    o = _oracle_fit(wl, generations=3, seed=4, want_pop=True)
    same = np.all(g["final_pop"] == o["final_pop"].astype(np.float32), axis=-1)
    observed("identical members (bar > 0.98)", round(float(same.mean()), 4))
    assert same.mean() > 0.98, same.mean()
    assert np.max(np.abs(g["final_fit"] - o["final_fit"]) / o["final_fit"]) < FIT_REL_TOL
    g = _gpu_fit(pt, wl, seed=4)
    o = _oracle_fit(wl, seed=4)
    # NP = 32 for 200 generations does not always collapse; compare where both sides agree on the optimum's RSS
    ok = np.abs(g["best_rss"] - o["best_rss"]) / o["best_rss"] < FIT_REL_TOL
    observed("blocks on the same optimum (bar >= 3)", ok.sum())
    assert ok.sum() >= 3, (g["best_rss"], o["best_rss"])
    assert np.max(np.abs(_wrap(g["best"][ok, 2] - o["best"][ok, 2]))) < PHI0_TOL
    assert np.max(np.abs(g["best"][ok, 3] - o["best"][ok, 3])) < F_TOL
    # every result is valid: its RSS is the oracle's objective at its own parameters
    chk = oracle.fitness(wl.x, wl.fs, g["best"][:, None, :].astype(np.float32))[:, 0]
    assert np.max(np.abs(chk - g["best_rss"]) / chk) < FIT_REL_TOL


def test_streamed_needs_workspace(pt, no_cluster):
    import ctypes as C
    L = pt.lib()
    cfg = pt.make_config(D=5, NP=32, generations=1, t0=-0.5)
    need = L.pt_fit_blocks_workspace_bytes(2, 65536, C.byref(cfg))
    assert need == 2 * 65536 * 4          # pt_run_kernel: one fp32 row per CTA (aligned copy of an unaligned / quantised block)
    with _forced_kernel("classic"):
        assert L.pt_fit_blocks_workspace_bytes(2, 65536, C.byref(cfg)) == 2 * 65536 * 4 * 2      # + the reference-phase row
    x = torch.zeros((2, 65536), dtype=torch.float32, device="cuda")
    box = torch.zeros((2, 5), dtype=torch.float64, device="cuda")
    best = torch.empty((2, 5), dtype=torch.float64, device="cuda")
    rss = torch.empty(2, dtype=torch.float32, device="cuda")
    st = torch.empty(2, dtype=torch.int32, device="cuda")
    rc = L.pt_fit_blocks(x.data_ptr(), 2, 65536, 65536.0, box.data_ptr(), box.data_ptr(), None, C.byref(cfg), best.data_ptr(),
                         rss.data_ptr(), st.data_ptr(), None, None, None, 0, None)
    assert rc == -2 and b"workspace" in L.pt_last_error_string()


# ----------------------------------------------------------------------------------------------
# cluster path: K CTAs of a thread-block cluster fit one block together
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [1, 2, 4, 8])
def test_fitness_cluster_sizes(pt, K):
    """Every cluster size against the oracle: slices of whole chunks, a ragged last slice (config 1: 78 chunks + 16
    samples), D = 6, NP not a multiple of the register blocking, and blocks with fewer chunks than CTAs."""
    with _forced_cluster(K):
        cfg = pt.make_config(D=5, NP=100, generations=1, seed=0, t0=-0.5)
        assert pt.pt_fit_blocks_plan(3, 10000, cfg)["cluster"] == K
        assert _fitness_case(pt, W.config1(blocks=[0, 30, 59]), NP=100) < FIT_REL_TOL
        assert _fitness_case(pt, W.config2(blocks=[5, 3000]), NP=128) < FIT_REL_TOL
        assert _fitness_case(pt, W.config3(blocks=[17900, 18000]), NP=36) < FIT_REL_TOL
        assert _fitness_case(pt, W.config0(cases=range(3)), NP=60) < FIT_REL_TOL
        wl = W.single_tone_blocks(range(2), 130, 130.0, config=4, f_range=(6.5, 26.0))    # 2 chunks: K capped at 2
        assert _fitness_case(pt, wl, NP=7) < FIT_REL_TOL
        wl = W.single_tone_blocks(range(2), 1002, 1002.0, config=4, f_range=(50, 200))    # unaligned rows: no bulk copy
        assert _fitness_case(pt, wl, NP=16) < FIT_REL_TOL


def test_cluster_plan_is_automatic_for_few_blocks(pt):
    cfg = pt.make_config(D=5, NP=100, generations=1000, seed=0, t0=-0.5)
    big = pt.pt_fit_blocks_plan(4, 65536, cfg)                         # 8 slices of 8192 samples: resident, not streamed
    assert big["cluster"] == 8 and big["resident"] == 1
    wl = W.config4(65536, 32, B=4)
    assert _fitness_case(pt, wl, NP=32, seed=1) < FIT_REL_TOL
    assert pt.pt_fit_blocks_plan(60, 10000, cfg)["cluster"] == 2       # BASELINE config 1: 60 blocks on 148 SMs
    assert pt.pt_fit_blocks_plan(1, 10000, cfg)["cluster"] == 8
    assert pt.pt_fit_blocks_plan(3600, 16000, cfg)["cluster"] == 1
    assert pt.pt_fit_blocks_plan(1, 256, cfg)["cluster"] == 1          # two chunks: not worth splitting


@pytest.mark.parametrize("K", [2, 8])
def test_fit_cluster_follows_the_oracle(pt, K):
    """The DE step is replicated in every CTA of the cluster and only partial sums are exchanged: the first generations
    are the oracle's trajectory member by member, and the full fit lands on the oracle's optimum."""
    with _forced_cluster(K):
        wl = W.config1(blocks=[0, 7, 33])
        g = _gpu_fit(pt, wl, generations=3, seed=9, want_pop=True)
        o = _oracle_fit(wl, generations=3, seed=9, want_pop=True)
        same = np.all(g["final_pop"] == o["final_pop"].astype(np.float32), axis=-1)
        observed("identical members (bar > 0.98)", round(float(same.mean()), 4))
        assert same.mean() > 0.98, same.mean()
        assert np.max(np.abs(g["final_fit"] - o["final_fit"]) / o["final_fit"]) < FIT_REL_TOL
        wl = W.config0(cases=range(5))
        g = _gpu_fit(pt, wl, seed=3)
        o = _oracle_fit(wl, seed=3)
        _check_fit_vs_oracle_and_truth(wl, g, o)


def test_fit_cluster_persistent_loop_and_single_cta_agree(pt):
    """More blocks than resident clusters (each cluster loops over several blocks) and the same blocks without
    clusters: same optimum; the sums differ only in fp32 rounding order."""
    wl = W.config1(blocks=range(40), generations=400)
    with _forced_cluster(8):
        a = _gpu_fit(pt, wl, seed=4)
    with _forced_cluster(1):
        b = _gpu_fit(pt, wl, seed=4)
    ok = ((a["status"] & 2) == 0) & ((b["status"] & 2) == 0)         # both populations collapsed
    observed("blocks on the same optimum (bar >= 36)", ok.sum())
    assert ok.sum() >= 36, ok.sum()
    assert np.max(np.abs(a["best_rss"][ok] - b["best_rss"][ok]) / b["best_rss"][ok]) < 1e-5
    assert np.max(np.abs(_wrap(a["best"][ok, 2] - b["best"][ok, 2]))) < PHI0_TOL
    assert np.max(np.abs(a["best"][ok, 3] - b["best"][ok, 3])) < F_TOL
    # every result is valid: its RSS is the oracle's objective at its own parameters
    chk = oracle.fitness(wl.x, wl.fs, a["best"][:, None, :].astype(np.float32))[:, 0]
    assert np.max(np.abs(chk - a["best_rss"]) / chk) < FIT_REL_TOL


def test_tail_wave_is_fitted_by_clusters_and_matches_the_single_launch(pt):
    """B = one full wave + a few blocks: the full wave runs on single CTAs, the remainder on clusters (second launch).  Same
    blocks with PT_CLUSTER=1 (one launch, no clusters): the Philox streams depend on the block index only, so the
    first generations are identical populations and the outputs land in the right rows."""
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    cfg = pt.make_config(D=5, NP=32, generations=2, seed=6, t0=-0.5)
    cps = pt.pt_fit_blocks_plan(100 * sms, 2048, cfg)["ctas_per_sm"]          # several CTAs per SM for blocks this short
    B = sms * cps + 5
    wl = W.config4(2048, 32, B=B, generations=2)
    cfg = pt.make_config(D=5, NP=32, generations=2, seed=6, t0=wl.t0)
    plan = pt.pt_fit_blocks_plan(B, 2048, cfg)
    assert plan["ctas_per_sm"] == cps and plan["grid"] == sms * cps, plan
    assert plan["cluster"] == 1 and plan["tail_cluster"] >= 2, plan       # 5 blocks of 2048 samples: clusters of 4 (two runs per CTA)
    a = _gpu_fit(pt, wl, generations=2, seed=6, want_pop=True)
    with _forced_cluster(1):
        b = _gpu_fit(pt, wl, generations=2, seed=6, want_pop=True)
    same = np.all(a["final_pop"] == b["final_pop"], axis=-1)
    observed("identical members (bar > 0.99)", round(float(same.mean()), 4))
    assert same.mean() > 0.99
    assert np.max(np.abs(a["final_fit"] - b["final_fit"]) / b["final_fit"]) < 1e-5
    k = 7          # the 5 tail blocks and the last 2 of the full wave, against the oracle
    o = oracle.fit_blocks(wl.x[-k:], wl.fs, wl.lo[-k:], wl.hi[-k:], NP=32, generations=2, F=wl.de["F"], CR=wl.de["CR"], seed=6,
                          block_index=wl.block_index[-k:], want_pop=True)
    assert np.max(np.abs(a["final_fit"][-k:] - o["final_fit"]) / o["final_fit"]) < FIT_REL_TOL
    assert (np.all(a["final_pop"][-k:] == o["final_pop"].astype(np.float32), axis=-1)).mean() > 0.98


# ----------------------------------------------------------------------------------------------
# DE trajectories
# ----------------------------------------------------------------------------------------------
def _gpu_fit(pt, wl, *, generations=None, seed=0, want_pop=False, F=None, CR=None, NP=None):
    de = dict(wl.de)
    cfg = pt.make_config(D=de["D"], NP=NP or de["NP"], generations=de["generations"] if generations is None else generations,
                         F=de["F"] if F is None else F, CR=de["CR"] if CR is None else CR, seed=seed, t0=wl.t0)
    r = pt.pt_fit_blocks(_cuda(wl.x), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg,
                         block_index=_cuda(wl.block_index.astype(np.int32)), want_pop=want_pop)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in r.items()}


def _oracle_fit(wl, *, generations=None, seed=0, want_pop=False, F=None, CR=None, NP=None):
    de = wl.de
    return oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=NP or de["NP"],
                             generations=de["generations"] if generations is None else generations,
                             F=de["F"] if F is None else F, CR=de["CR"] if CR is None else CR, seed=seed,
                             block_index=wl.block_index, want_pop=want_pop)


def test_generation_zero_population_and_fitness(pt):
    wl = W.config0(cases=range(4))
    g = _gpu_fit(pt, wl, generations=0, seed=5, want_pop=True)
    o = _oracle_fit(wl, generations=0, seed=5, want_pop=True)
    assert np.array_equal(g["final_pop"], o["final_pop"].astype(np.float32))
    assert np.max(np.abs(g["final_fit"] - o["final_fit"]) / o["final_fit"]) < FIT_REL_TOL
    assert np.max(np.abs(g["best_rss"] - o["best_rss"]) / o["best_rss"]) < FIT_REL_TOL
    assert np.array_equal(g["best"], o["best"])            # fp64 best is the fp64 member itself


@pytest.mark.parametrize("D", [5, 6])
def test_first_generations_follow_the_oracle_trajectory(pt, D):
    """Mutation, crossover and bound handling run in fp64 without contraction, so until a selection decision
    falls inside the fp32 fitness error the GPU population IS the oracle population."""
    wl = W.config0(cases=range(4)) if D == 5 else W.config3(blocks=[17990, 18010], NP=60, generations=5)
    for G, F, CR in ((1, 0.5, 0.9), (4, 1.7, 0.6)):
        g = _gpu_fit(pt, wl, generations=G, seed=21, want_pop=True, F=F, CR=CR, NP=60)
        o = _oracle_fit(wl, generations=G, seed=21, want_pop=True, F=F, CR=CR, NP=60)
        same = np.all(g["final_pop"] == o["final_pop"].astype(np.float32), axis=-1)
        observed("identical members (bar > 0.98)", round(float(same.mean()), 4))
        assert same.mean() > 0.98, same.mean()
        assert np.all(g["final_pop"] >= wl.lo[:, None, :].astype(np.float32) - 1e-6)
        assert np.all(g["final_pop"] <= wl.hi[:, None, :].astype(np.float32) + 1e-6)


def _check_fit_vs_oracle_and_truth(wl, g, o, n_sigma=4.0, extra_f_bias=None):
    D = wl.D
    dphi = _wrap(g["best"][:, 2] - o["best"][:, 2])
    df = g["best"][:, 3] - o["best"][:, 3]
    assert np.max(np.abs(dphi)) < PHI0_TOL, np.max(np.abs(dphi))
    assert np.max(np.abs(df)) < F_TOL, np.max(np.abs(df))
    assert np.max(np.abs(g["best_rss"] - o["best_rss"]) / o["best_rss"]) < FIT_REL_TOL
    assert np.max(np.abs(g["best"][:, 0] - o["best"][:, 0])) < 1e-3
    for k in range(wl.B):
        sig = wl.meta["sigma_per_block"][k] if "sigma_per_block" in wl.meta else wl.sigma
        sd = _crlb(wl.truth[k], wl.N, wl.fs, sig, D)
        for res in (g, o):
            # well-determined combinations: phi0 and f where the box is wide enough for the
            # optimum to be interior; a face-pinned optimum is judged against the oracle only
            if res["status"][k] & 1:
                continue
            bias_f = 0.0 if extra_f_bias is None else extra_f_bias[k]
            assert abs(_wrap(res["best"][k, 2] - wl.truth[k, 2])) < n_sigma * sd[2] + 1e-3
            assert abs(res["best"][k, 3] - wl.truth[k, 3] - bias_f) < n_sigma * sd[3]


def test_fit_config0_32_seeds(pt):
    """BASELINE config 0: NP = 60, D = 5, F = 0.5, CR = 0.9, 500 generations, box +-20 % around truth."""
    wl = W.config0(cases=range(32))
    g = _gpu_fit(pt, wl, seed=3)
    o = _oracle_fit(wl, seed=3)
    _check_fit_vs_oracle_and_truth(wl, g, o)
    # status bit0 (best on a box face) is decided by the same rule on both sides, but the fp32 objective cannot
    # resolve the last 1e-6 (hi-lo) of the approach to a face: the GPU flag implies the
    # oracle's, and where the oracle sits on a face the GPU's best is next to the same face
    assert np.all((g["status"] & 1) <= (o["status"] & 1))
    w = wl.hi - wl.lo
    on_face = np.minimum(o["best"] - wl.lo, wl.hi - o["best"]) <= 1e-6 * w
    near = np.minimum(g["best"] - wl.lo, wl.hi - g["best"]) <= 5e-3 * w
    assert np.all(near[on_face])
    assert np.all((g["status"] & 2) == 0) and np.all((o["status"] & 2) == 0)
    # noiseless: both recover the generating truth
    wn = W.config0(cases=range(4), noiseless=True)
    gn = _gpu_fit(pt, wn, seed=3)
    assert np.max(np.abs(_wrap(gn["best"][:, 2] - wn.truth[:, 2]))) < 1e-4
    assert np.max(np.abs(gn["best"][:, 3] - wn.truth[:, 3])) < 1e-5
    assert np.max(gn["best_rss"]) < 1e-6


def test_fit_config0_paper_box_and_table4_settings(pt):
    """Robustness cases: paper-style box (phi0 in [-pi, pi]) and Table 4's F = 0.5, CR = 0.85, 200 its."""
    wl = W.config0(cases=range(8), box="paper")
    g = _gpu_fit(pt, wl, seed=8)
    o = _oracle_fit(wl, seed=8)
    _check_fit_vs_oracle_and_truth(wl, g, o)
    wl = W.config0(cases=range(8))
    g = _gpu_fit(pt, wl, seed=9, generations=200, CR=0.85)
    o = _oracle_fit(wl, seed=9, generations=200, CR=0.85)
    _check_fit_vs_oracle_and_truth(wl, g, o)


def test_fit_config1_blocks(pt):
    """Config 1 (N = 10000, NP = 100, 1000 generations) on three blocks; D = 5 on a cubic-frequency signal is
    biased by T^2 f''/40."""
    wl = W.config1(blocks=[0, 30, 59])
    g = _gpu_fit(pt, wl, seed=2)
    o = _oracle_fit(wl, seed=2)
    bias = wl.T**2 * wl.meta["fddot_true"] / 40.0
    assert np.all((g["status"] & 2) == 0) and np.all((o["status"] & 2) == 0)
    _check_fit_vs_oracle_and_truth(wl, g, o, extra_f_bias=bias)


def test_fit_config1_block59_premature_convergence_is_a_valid_result_on_both_sides(pt):
    """DE is a heuristic and the two sides follow the same trajectory only until a selection decision falls inside
    the fp32 fitness error.  Known hard case: block 59 of config 1 (a +-278 Hz box searched for a 1 Hz wide lobe).
    With seed 1 the ORACLE's population collapses early (a0 = 0.960, chi^2 = 512.49) while seeds 2-4 reach the
    optimum (a0 = 1.004, chi^2 = 502.60); the paper's remedy for a doubtful block is to search again.
    Several results are correct here, so: every run must be a VALID result (its chi^2 is the oracle's objective at
    its own parameters, inside the box), both sides must reach the lowest optimum for at least one seed, and all
    runs that reach it must agree at the parity bounds."""
    wl = W.config1(blocks=[59])
    runs = {}
    for seed in (1, 2, 3):
        runs[("oracle", seed)] = _oracle_fit(wl, seed=seed)
        runs[("gpu", seed)] = _gpu_fit(pt, wl, seed=seed)
    rss = {}
    for k, v in runs.items():
        rss[k] = float(v["best_rss"][0])
        r = oracle.rss(wl.x[0], wl.fs, v["best"][0])
        assert abs(rss[k] - r) / r < FIT_REL_TOL, k
        assert np.all(v["best"][0] >= wl.lo[0]) and np.all(v["best"][0] <= wl.hi[0]), k
    lowest = min(rss.values())
    at_optimum = [k for k in runs if rss[k] - lowest < FIT_REL_TOL * lowest]
    assert any(k[0] == "oracle" for k in at_optimum) and any(k[0] == "gpu" for k in at_optimum), rss
    ref = runs[[k for k in at_optimum if k[0] == "oracle"][0]]["best"][0]
    for k in at_optimum:
        assert abs(_wrap(runs[k]["best"][0, 2] - ref[2])) < PHI0_TOL, (k, rss)
        assert abs(runs[k]["best"][0, 3] - ref[3]) < F_TOL, (k, rss)
        assert abs(runs[k]["best"][0, 0] - ref[0]) < 1e-3, (k, rss)


def test_fit_config2_blocks(pt):
    wl = W.config2(blocks=[0, 1800])
    g = _gpu_fit(pt, wl, seed=2)
    o = _oracle_fit(wl, seed=2)
    _check_fit_vs_oracle_and_truth(wl, g, o)


def test_fit_config3_blocks(pt):
    """D = 6, T = 0.1 s: fdot / fddot / a1 are not observable -- parity is required on
    phi0, f, a0 and the block phase increment only."""
    wl = W.config3(blocks=[100, 17950])
    g = _gpu_fit(pt, wl, seed=4)
    o = _oracle_fit(wl, seed=4)
    dphi = _wrap(g["best"][:, 2] - o["best"][:, 2])
    assert np.max(np.abs(dphi)) < PHI0_TOL
    # north_star's |df| < 1e-3 Hz holds as it stands on blocks at the configured SNR (block 100; measured on 95 + 25 blocks in
    # tests/test_gpu_oracle_subset.py).  Block 17950 sits at the bottom of the amplitude fade (a0 = 0.105, -10 dB per sample):
    # there the chi^2 surface is flatter than the fp32 objective resolves and the bar is max(1e-3 Hz, 0.01 sigma_f) (R20).
    T = wl.T
    for k in range(wl.B):
        sig_f = _crlb(wl.truth[k], wl.N, wl.fs, wl.meta["sigma_per_block"][k] if "sigma_per_block" in wl.meta else wl.sigma, 6)[3]
        f_tol = F_TOL if wl.truth[k, 0] >= 0.3 else max(F_TOL, 0.01 * sig_f)
        assert abs(g["best"][k, 3] - o["best"][k, 3]) < f_tol, (k, f_tol)
        inc_g = 2 * np.pi * (g["best"][k, 3] * T + g["best"][k, 5] * T**3 / 24)
        inc_o = 2 * np.pi * (o["best"][k, 3] * T + o["best"][k, 5] * T**3 / 24)
        assert abs(inc_g - inc_o) < 2 * np.pi * f_tol * T + 1e-6
    assert np.max(np.abs(g["best_rss"] - o["best_rss"]) / o["best_rss"]) < FIT_REL_TOL


def test_zero_width_box_and_tiny_population(pt):
    wl = W.config0(cases=range(2))
    lo, hi = wl.lo.copy(), wl.hi.copy()
    lo[:, 1] = hi[:, 1] = wl.truth[:, 1]        # a1 fixed
    lo[1] = hi[1] = wl.truth[1]                 # block 1: every coordinate fixed
    wl.lo, wl.hi = lo, hi
    g = _gpu_fit(pt, wl, seed=6, NP=4, generations=30, want_pop=True)
    o = _oracle_fit(wl, seed=6, NP=4, generations=30, want_pop=True)
    assert np.all(g["best"][:, 1] == wl.truth[:, 1])
    assert np.array_equal(g["best"][1], wl.truth[1])
    assert g["status"][1] == 0 and o["status"][1] == 0
    assert np.all(g["final_pop"][1] == wl.truth[1].astype(np.float32))
    assert abs(g["best_rss"][1] - o["best_rss"][1]) / o["best_rss"][1] < FIT_REL_TOL


def test_status_face_bit(pt):
    wl = W.config0(cases=[1])
    wl.lo[0, 3] = wl.truth[0, 3] + 0.05
    wl.hi[0, 3] = wl.truth[0, 3] + 0.5
    g = _gpu_fit(pt, wl, seed=3, NP=40, generations=300)
    assert g["status"][0] & 1
    assert abs(g["best"][0, 3] - wl.lo[0, 3]) <= 1e-6 * 0.45
    g2 = _gpu_fit(pt, W.config0(cases=[2]), seed=3, NP=32, generations=2)
    assert g2["status"][0] & 2                   # not collapsed after two generations


def test_block_index_selects_the_stream_and_persistent_loop_is_consistent(pt):
    """More blocks than resident CTAs: every CTA loops over several blocks; results must equal a one-block run."""
    wl = W.single_tone_blocks(range(700), 256, 256.0, config=4, f_range=(20, 60))
    wl.de = dict(NP=16, D=5, generations=12, F=0.5, CR=0.9)
    g = _gpu_fit(pt, wl, seed=77, want_pop=True)
    for k in (0, 299, 699):
        sub = W.single_tone_blocks([k], 256, 256.0, config=4, f_range=(20, 60))
        sub.de = wl.de
        sub.block_index = np.array([k], dtype=np.uint32)
        gk = _gpu_fit(pt, sub, seed=77, want_pop=True)
        assert np.array_equal(gk["final_pop"][0], g["final_pop"][k])
        assert np.array_equal(gk["best"][0], g["best"][k])
    o = oracle.fit_blocks(wl.x[:5], wl.fs, wl.lo[:5], wl.hi[:5], NP=16, generations=12, seed=77, want_pop=True)
    same = np.all(g["final_pop"][:5] == o["final_pop"].astype(np.float32), axis=-1)
    observed("identical members (bar > 0.9)", round(float(same.mean()), 4))
    assert same.mean() > 0.9


# ----------------------------------------------------------------------------------------------
# Doppler products
# ----------------------------------------------------------------------------------------------
def _compare_products(pt, best, T, los, m):
    pb_o, tot_o, iv_o = oracle.doppler_products(best, T, los, m)
    pb, tot, iv = pt.pt_doppler_products(_cuda(best), T, los, m)
    pb, tot = pb.cpu().numpy(), tot.cpu().numpy()
    assert np.isnan(pb[-1, 8]) and np.isnan(pb[-1, 9])
    # phases mod 2 pi and wrapped residuals carry the absolute rounding of a phase of magnitude |phi|
    scale = np.maximum(np.abs(pb_o), 1.0)
    scale[:, [3, 4, 8]] = np.maximum(np.abs(pb_o[:, [7]]), 1.0)
    err = np.abs(pb - pb_o) / scale
    assert np.nanmax(err) < 1e-9
    assert np.max(np.abs(tot - tot_o) / np.maximum(np.abs(tot_o), 1.0)) < 1e-9
    for a, b in zip(iv, iv_o):
        a = a.cpu().numpy()
        assert a.shape == b.shape
        if b.size:
            assert np.max(np.abs(a - b) / np.maximum(np.abs(b), 1.0)) < 1e-9


@pytest.mark.parametrize("B,D,T", [(1, 5, 1.0), (60, 5, 1.0), (3600, 5, 1.0), (36000, 6, 0.1), (100003, 6, 0.5)])
def test_doppler_products_vs_oracle(pt, B, D, T):
    rng = np.random.default_rng(B)
    best = np.stack([rng.uniform(0.5, 1.5, B), rng.uniform(-0.1, 0.1, B), rng.uniform(-np.pi, np.pi, B),
                     rng.uniform(1000, 5200, B), rng.uniform(-5, 5, B)] + ([rng.uniform(-1, 1, B)] if D == 6 else []),
                    axis=1)
    m = [max(1, int(round(tc / T))) for tc in (1.0, 10.0, 60.0)]
    _compare_products(pt, best, T, 0.031, m)


def test_doppler_products_appendix_a(pt, golden_dir):
    """The paper's worked example through the CUDA path."""
    from test_oracle_doppler import _read_appendix, _theta_from_paper_units
    blocks, borders, _ = _read_appendix(golden_dir)
    best = np.array([_theta_from_paper_units(r) for r in blocks])
    pb, tot, _ = pt.pt_doppler_products(_cuda(best), 2.0)
    pb = pb.cpu().numpy()
    assert np.all(np.abs(pb[:, 7] - blocks[:, 7]) <= 1.5e-3)
    assert np.all(np.abs(pb[:-1, 6] - borders[:, 2]) <= 3e-3)
    assert np.all(np.abs(pb[1:, 5] - borders[:, 4]) <= 3e-3)
    assert np.all(np.abs(_wrap(pb[1:, 3] - borders[:, 3])) <= 2.5e-3)


# ----------------------------------------------------------------------------------------------
# host-buffer entry point and integrated phase
# ----------------------------------------------------------------------------------------------
def test_track_host_equals_device_path_and_integrated_phase_config1(pt):
    """Config 1 at full size (60 x 10000, NP = 100, 1000 generations) through pt_track_host; the 60 s integrated
    phase is compared with the analytic integral minus the D = 5 truncation term."""
    wl = W.config1()
    cfg = pt.make_config(D=5, NP=100, generations=1000, seed=1, t0=wl.t0)
    h = pt.pt_track_host(torch.from_numpy(wl.x), wl.fs, torch.from_numpy(wl.lo), torch.from_numpy(wl.hi), cfg, 0.0,
                         [1, 10, 60])
    g = _gpu_fit(pt, wl, seed=1)
    assert np.array_equal(h["best"].numpy(), g["best"])
    pb, tot, iv = pt.pt_doppler_products(_cuda(g["best"]), wl.T, 0.0, [1, 10, 60])
    assert np.array_equal(h["total_phase"].numpy(), tot.cpu().numpy())
    assert np.array_equal(h["intervals"][2].numpy(), iv[2].cpu().numpy())
    phi60 = h["intervals"][2].numpy()[0, 0]
    analytic = wl.meta["dphi_true"].sum()
    trunc = np.sum(2 * np.pi * wl.meta["fddot_true"] * wl.T**3 / 60.0)
    assert abs(phi60 - (analytic - trunc)) < 0.34          # 4 sqrt(60) sigma(dphi_block), SURVEY q16
    assert abs(phi60 - iv[1].cpu().numpy()[:, 0].sum()) < 1e-6
    # oracle products on the GPU's parameters
    pb_o, tot_o, _ = oracle.doppler_products(g["best"], wl.T, 0.0, [1, 10, 60])
    assert abs(tot_o[-1] - phi60) < 1e-6
    # three of the blocks against the oracle's own fit
    sub = W.config1(blocks=[7, 41])
    o = _oracle_fit(sub, seed=1)
    assert np.max(np.abs(_wrap(g["best"][[7, 41], 2] - o["best"][:, 2]))) < PHI0_TOL
    assert np.max(np.abs(g["best"][[7, 41], 3] - o["best"][:, 3])) < F_TOL


def test_full_size_config2_sampled_blocks(pt):
    """BASELINE config 2 at full size in bench.py's launch configuration (3600 x 16000, NP = 128, 1000 generations):
    sampled blocks are checked one by one with the oracle's objective; properties are checked on all blocks."""
    wl = W.config2()
    g = _gpu_fit(pt, wl, seed=1)
    assert np.all(np.isfinite(g["best"])) and np.all(np.isfinite(g["best_rss"]))
    assert np.all(g["best"] >= wl.lo) and np.all(g["best"] <= wl.hi)
    assert np.all((g["status"] & 2) == 0)                              # every population collapsed (1e-3 rule)
    # chi^2 at the optimum is the summed noise power: (N - D) sigma^2 within 5 sigma, all blocks
    z = (g["best_rss"] - (wl.N - 5) * wl.sigma**2) / (wl.sigma**2 * np.sqrt(2.0 * wl.N))
    assert np.max(np.abs(z)) < 5.0 and abs(z.mean()) < 0.2
    for k in range(0, 3600, 240):
        r_or = oracle.rss(wl.x[k], wl.fs, g["best"][k])               # oracle's objective at the GPU's optimum
        assert abs(g["best_rss"][k] - r_or) / r_or < FIT_REL_TOL
        assert r_or <= oracle.rss(wl.x[k], wl.fs, wl.truth[k])        # at least as good as the generating truth
    # border continuity (Eq. 8) at the noise level: phase residual sigma ~ 2 x 12 mrad x a few
    pb, tot, iv = pt.pt_doppler_products(_cuda(g["best"]), wl.T, 0.0, [1, 10, 60])
    pb = pb.cpu().numpy()
    assert np.nanstd(pb[:, 8]) < 0.1
    # 60-s integration Doppler against the analytic phase advance (truncation <= 1.3e-3 rad per 60 s)
    phi60 = iv[2].cpu().numpy()[:, 0]
    true60 = wl.meta["dphi_true"].reshape(60, 60).sum(axis=1)
    sd_f = _crlb(wl.truth[1800], wl.N, wl.fs, wl.sigma, 5)[3]
    sd60 = np.sqrt(60.0) * 2 * np.pi * sd_f * wl.T            # Eq. 17: sum of 60 independent block increments
    assert np.max(np.abs(phi60 - true60)) < 4.5 * sd60
    assert np.std(phi60 - true60) < 1.5 * sd60
    # one sampled block against the oracle's own DE fit
    sub = W.config2(blocks=[1234])
    o = _oracle_fit(sub, seed=1)
    assert abs(_wrap(g["best"][1234, 2] - o["best"][0, 2])) < PHI0_TOL
    assert abs(g["best"][1234, 3] - o["best"][0, 3]) < F_TOL


def test_full_size_config3_sampled_blocks(pt):
    """BASELINE config 3 at full size in bench.py's launch configuration (36000 x 10000 samples, NP = 128, D = 6, 1500
    generations; the tensor-core kernel, two blocks per CTA, tail wave on clusters): properties on all blocks, sampled blocks
    one by one with the oracle's objective, and one sampled block against the oracle's own DE fit."""
    wl = W.config3()
    g = _gpu_fit(pt, wl, seed=1)
    assert np.all(np.isfinite(g["best"])) and np.all(np.isfinite(g["best_rss"]))
    assert np.all(g["best"] >= wl.lo) and np.all(g["best"] <= wl.hi)
    assert np.all((g["status"] & (2 | 8 | 16)) == 0)                  # collapsed, finite, boxes in order
    # chi^2 at the optimum is the summed noise power: (N - D) sigma^2 within 5 sigma on all blocks
    # -- where the box leaves the optimum free.  The literal box is +-20 % of |theta|: where the true phi0 happens to
    # be within ~0.1 rad of zero its box is narrower than the noise moves the least-squares phase (4.7 mrad at 10 dB), the fit is
    # a CONSTRAINED optimum and its chi^2 is larger (measured: 4 of 36000 blocks with z = 5.9 .. 8.7, all with |phi0_true| < 0.02):
    # there only the lower side is asserted.
    z = (g["best_rss"] - (wl.N - 6) * wl.sigma**2) / (wl.sigma**2 * np.sqrt(2.0 * wl.N))
    free = np.abs(wl.truth[:, 2]) > 0.15
    assert np.max(np.abs(z[free])) < 5.5 and abs(z[free].mean()) < 0.1
    assert np.min(z) > -5.5 and np.mean(z > 5.5) < 1e-3
    for k in range(0, 36000, 1500):
        r_or = oracle.rss(wl.x[k], wl.fs, g["best"][k])
        assert abs(g["best_rss"][k] - r_or) / r_or < FIT_REL_TOL
        assert r_or <= oracle.rss(wl.x[k], wl.fs, wl.truth[k]) * (1 + 1e-9)
    # Eq. 16-17: the 60-s integrated phase against the analytic phase advance; sigma of a block's increment from the
    # Cramer-Rao bound of f (unfaded blocks; the fade around t = 1800 s is excluded from the bound, not from the sum)
    pb, tot, iv = pt.pt_doppler_products(_cuda(g["best"]), wl.T, 0.0, [10, 100, 600])
    phi60 = iv[2].cpu().numpy()[:, 0]
    true60 = wl.meta["dphi_true"].reshape(60, 600).sum(axis=1)
    sd_f = _crlb(wl.truth[100], wl.N, wl.fs, wl.sigma, 6)[3]
    sd60 = np.sqrt(600.0) * 2 * np.pi * sd_f * wl.T
    clear = np.ones(60, dtype=bool)
    clear[27:33] = False                                               # 1620 .. 1980 s: the faded minutes
    assert np.max(np.abs(phi60 - true60)[clear]) < 5.0 * sd60
    sub = W.config3(blocks=[23456])
    o = _oracle_fit(sub, seed=1)
    assert abs(_wrap(g["best"][23456, 2] - o["best"][0, 2])) < PHI0_TOL
    assert abs(g["best"][23456, 3] - o["best"][0, 3]) < F_TOL
