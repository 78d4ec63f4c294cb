"""Parity run order step (3) of SURVEY.md 8(d) on the oracle subsets: pt_fit_blocks vs the oracle's own DE fit on blocks 0-59 plus
every 100th (config 2) / 1000th (config 3) block, at the north_star bars |dphi0| < 5 mrad and |df| < 1e-3 Hz.  The oracle runs all
generations (about 3 minutes per config on 16 host cores).  Observed figures are PRINTED (run with -s) and pinned, so that a
regression of the fraction of blocks on the same optimum, or of the margins, is visible.

DE is a heuristic (R19): on a +-20 % frequency box a run can converge prematurely on EITHER side (config 2, seed 1:
block 40 on the GPU, block 46 in the oracle).  Parameters are compared where both sides reached the same optimum (RSS within
1e-4 relative); every other result must still be VALID: its RSS is the oracle's objective at its own parameters, inside the box."""
import numpy as np
import pytest

import oracle
from paper_1906_10598_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

PHI0_TOL, F_TOL, FIT_REL_TOL = 5e-3, 1e-3, 1e-4


@pytest.fixture(scope="module")
def pt():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device; there is no CPU fallback")
    from paper_1906_10598_b200 import pt as _pt
    _pt.lib()
    return _pt


def _wrap(d):
    return (np.asarray(d) + np.pi) % (2 * np.pi) - np.pi


def _both(pt, wl, seed=1):
    de = wl.de
    cfg = pt.make_config(D=de["D"], NP=de["NP"], generations=de["generations"], F=de["F"], CR=de["CR"], seed=seed, t0=wl.t0)
    r = pt.pt_fit_blocks(torch.from_numpy(wl.x).cuda(), wl.fs, torch.from_numpy(wl.lo).cuda(), torch.from_numpy(wl.hi).cuda(), cfg,
                         block_index=torch.from_numpy(wl.block_index.astype(np.int32)).cuda())
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in r.items()}
    o = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=de["NP"], generations=de["generations"], F=de["F"], CR=de["CR"], seed=seed,
                          block_index=wl.block_index)
    return g, o


def _sigma_f(wl, k):
    """Cramer-Rao 1-sigma of f for block k (Fisher matrix of Eq. 2 at the generating truth, white noise of the workload)."""
    N, fs, D = wl.N, wl.fs, wl.de["D"]
    t = -N / (2 * fs) + np.arange(N) / fs
    th = list(wl.truth[k]) + [0.0] * (6 - D)
    ph = th[2] + 2 * np.pi * (th[3] * t + th[4] * t * t / 2 + th[5] * t**3 / 6)
    A = th[0] + th[1] * t
    c, s = np.cos(ph), np.sin(ph)
    J = [c, t * c, -A * s, -A * s * 2 * np.pi * t, -A * s * np.pi * t * t] + ([-A * s * np.pi * t**3 / 3] if D == 6 else [])
    J = np.array(J)
    return float(np.sqrt(np.diag(np.linalg.inv(J @ J.T / wl.sigma**2)))[3])


def _report_and_check(name, wl, g, o, min_same, f_tol=None):
    dphi = _wrap(g["best"][:, 2] - o["best"][:, 2])
    df = g["best"][:, 3] - o["best"][:, 3]
    drss = (g["best_rss"] - o["best_rss"]) / o["best_rss"]
    same = np.abs(drss) < FIT_REL_TOL
    q = lambda v: tuple(float(x) for x in np.quantile(np.abs(v[same]), [0.5, 0.9, 0.99, 1.0]))
    print("\n[%s] %d blocks: same optimum on %d (%.1f %%); |dphi0| rad 50/90/99/max %.2e %.2e %.2e %.2e; |df| Hz 50/90/99/max "
          "%.2e %.2e %.2e %.2e; max |dRSS|/RSS %.2e; off-optimum blocks %s" %
          ((name, wl.B, int(same.sum()), 100.0 * same.mean()) + q(dphi) + q(df) +
           (float(np.max(np.abs(drss[same]))), [int(b) for b in wl.block_index[~same]])))
    assert same.mean() >= min_same
    assert np.max(np.abs(dphi[same])) < PHI0_TOL
    f_tol = np.full(wl.B, F_TOL) if f_tol is None else f_tol
    assert np.all(np.abs(df[same]) < f_tol[same]), (df[same], f_tol[same])
    # every result, on either side, is a valid one: its objective value is the oracle's objective at its own parameters
    for k in np.nonzero(~same)[0]:
        for side in (g, o):
            r = oracle.rss(wl.x[k], wl.fs, side["best"][k])
            assert abs(float(side["best_rss"][k]) - r) / r < FIT_REL_TOL
            assert np.all(side["best"][k] >= wl.lo[k]) and np.all(side["best"][k] <= wl.hi[k])


def test_config2_oracle_subset(pt):
    """BASELINE config 2 (T = 1 s, 0 dB): 95 blocks.  Round 2 measurement (pt_run_kernel): 92/95 on the same optimum, |df| max 9.1e-5 Hz, |dphi0| max 2.5e-4 rad."""
    wl = W.config2(blocks=W.oracle_subset(2))
    g, o = _both(pt, wl)
    _report_and_check("config 2 oracle subset", wl, g, o, min_same=0.95)


def test_config3_oracle_subset(pt):
    """BASELINE config 3 (T = 0.1 s, D = 6, 10 dB, block 18000 sits at the bottom of the amplitude fade): 95 blocks at the
    north_star bar itself -- |df| < 1e-3 Hz, no relaxation.  Round 2 measurement (pt_run_kernel): 95/95 on the same optimum, |df| 50/90/99/max =
    1.2e-4 / 2.6e-4 / 3.5e-4 / 4.4e-4 Hz, |dphi0| max 7.0e-5 rad.  fdot / fddot / a1 are not observable at T = 0.1 s
    (reading R13) and are not compared."""
    wl = W.config3(blocks=W.oracle_subset(3))
    g, o = _both(pt, wl)
    _report_and_check("config 3 oracle subset", wl, g, o, min_same=0.97)
    T = wl.T
    inc_g = 2 * np.pi * (g["best"][:, 3] * T + g["best"][:, 5] * T**3 / 24)
    inc_o = 2 * np.pi * (o["best"][:, 3] * T + o["best"][:, 5] * T**3 / 24)
    assert np.max(np.abs(inc_g - inc_o)) < 2 * np.pi * F_TOL * T + 1e-6


def test_config3_fade_region(pt):
    """Config 3 through the amplitude fade (blocks 16800 .. 19200, every 100th; amplitude 1 -> 0.1 -> 1, i.e. 10 dB down to -10 dB
    per sample) at the north_star bar itself, |df| < 1e-3 Hz on every block, no relaxation.  With pt_run_kernel (objective summed
    in fp32 over a run, compensated across runs, fp64 from there on) the measured distribution is 25/25 blocks on the same optimum,
    |df| 50/90/99/max = 1.3e-4 / 4.4e-4 / 7.5e-4 / 8.1e-4 Hz.  (pt_block_kernel, whose objective is fp32 throughout, left one block --
    18100, a0 = 0.115 -- at 1.2e-3 Hz = 0.003 sigma_f; R20 keeps that measurement.)"""
    blocks = list(range(16800, 19201, 100))
    wl = W.config3(blocks=blocks)
    g, o = _both(pt, wl)
    _report_and_check("config 3 fade region", wl, g, o, min_same=0.95)
    df = np.abs(g["best"][:, 3] - o["best"][:, 3])
    print("[config 3 fade region] blocks with |df| >= 1e-3 Hz: %s" % [(int(b), float(v)) for b, v in zip(blocks, df) if v >= F_TOL])
