"""GPU parity of row f-1, first part: initial range determination by FFT acquisition (
DESIGN.md reading R24) -- pt_acquire through the C ABI against the fp64 numpy oracle, and the chain
pt_acquire -> pt_fit_blocks with no caller-supplied ranges.

Bars: peak bins bit-exact (integer decision; the fp32 transform's power error, ~1e-6 relative, is far below the
separation of a spectral peak from its neighbours on these inputs); refined frequencies within 1e-3 bin, amplitudes
within 1e-4 relative, boxes within the same bounds scaled by their definition.
"""
import numpy as np
import pytest

import oracle
from paper_1906_10598_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


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


def _compare(pt, wl, M, S, **kw):
    acq = pt.make_acq_config(M=M, spacing=S, **kw)
    g = {k: v.cpu().numpy() for k, v in pt.pt_acquire(_cuda(wl.x), wl.fs, wl.D, acq).items()}
    o = oracle.acquire(wl.x, wl.fs, wl.D, M, S, **kw)
    res = wl.fs / M
    assert np.array_equal(g["est"][:, 5:8], o["est"][:, 5:8])                      # peak bins
    assert np.max(np.abs(g["est"][:, 1:4] - o["est"][:, 1:4])) < 1e-3 * res        # refined frequencies
    assert np.max(np.abs(g["est"][:, 0] / o["est"][:, 0] - 1)) < 1e-4              # amplitude
    assert np.max(np.abs(g["est"][:, 4] - o["est"][:, 4])) < 1e-3 * res / (S / wl.fs)
    assert np.max(np.abs(g["lo"][:, 3] - o["lo"][:, 3])) < 1.2e-3 * res and np.max(np.abs(g["hi"][:, 3] - o["hi"][:, 3])) < 1.2e-3 * res
    for j in (0, 1):
        assert np.allclose(g["lo"][:, j], o["lo"][:, j], rtol=1e-4, atol=0) and np.allclose(g["hi"][:, j], o["hi"][:, j], rtol=1e-4, atol=0)
    assert np.array_equal(g["lo"][:, 2], o["lo"][:, 2]) and np.array_equal(g["hi"][:, 2], o["hi"][:, 2])
    assert np.max(np.abs(g["lo"][:, 4] - o["lo"][:, 4])) < 1e-3 * res / (S / wl.fs)
    if wl.D == 6:
        assert np.array_equal(g["lo"][:, 5], o["lo"][:, 5]) and np.array_equal(g["hi"][:, 5], o["hi"][:, 5])
    return g, o


@pytest.mark.parametrize("M", [64, 256, 512])
def test_acquire_config0(pt, M):
    wl = W.config0(cases=range(24))
    _compare(pt, wl, M, (wl.N - M) // 2)
    _compare(pt, wl, M, 100, f_rel=0.0, f_bins=2.0, fdot_bins=3.0, a_rel=0.25, a1_rel=0.5)


def test_acquire_tracks(pt):
    _compare(pt, W.config1(blocks=[0, 20, 40, 59]), 2048, 3900)
    _compare(pt, W.config2(blocks=[0, 900, 1800, 2700, 3599]), 4096, 5952)          # 0 dB per sample
    _compare(pt, W.config2(blocks=[5, 3000]), 8192, 3904)                           # largest piece (64 KB of shared memory)
    _compare(pt, W.config3(blocks=[0, 17000, 17990, 18010, 35999]), 2048, 3976)     # D = 6, through the fade
    # more blocks than resident CTAs: the persistent loop over blocks
    wl = W.config4(1024, 32, B=1500, generations=1)
    _compare(pt, wl, 256, 300)


def test_acquire_then_fit_needs_no_caller_ranges(pt):
    """The chain the paper runs at the start of a track: ranges from the FFT, then the DE fit inside them.  The paper's
    +-10 % of c1 on config 0; a two-bin range on config 2.  Fitted phi0 and f agree with the fit in the truth-centred
    boxes of the acceptance tests (same interior least-squares optimum) to the usual bars."""
    wl = W.config0(cases=range(8))
    acq = pt.make_acq_config(M=256, spacing=(wl.N - 256) // 2, a_rel=0.2)
    r = pt.pt_acquire(_cuda(wl.x), wl.fs, 5, acq)
    lo, hi = r["lo"].cpu().numpy(), r["hi"].cpu().numpy()
    assert np.all(lo[:, 3] <= wl.truth[:, 3]) and np.all(wl.truth[:, 3] <= hi[:, 3])
    cfg = pt.make_config(D=5, NP=80, generations=600, F=0.5, CR=0.9, seed=3, t0=wl.t0)
    g = {k: v.cpu().numpy() for k, v in pt.pt_fit_blocks(_cuda(wl.x), wl.fs, r["lo"], r["hi"], cfg).items()}
    # reference: the oracle's fit in the truth-centred "paper" box, whose optimum is interior like the one found here
    # (the +-20 % "literal" box pins a1 on a face on some of these blocks, a different constrained optimum)
    wp = W.config0(cases=range(8), box="paper")
    ref = oracle.fit_blocks(wp.x, wp.fs, wp.lo, wp.hi, NP=60, generations=500, F=0.5, CR=0.9, seed=3)
    assert np.max(np.abs(g["best_rss"] - ref["best_rss"]) / ref["best_rss"]) < 1e-4
    assert np.max(np.abs(_wrap(g["best"][:, 2] - ref["best"][:, 2]))) < 5e-3
    assert np.max(np.abs(g["best"][:, 3] - ref["best"][:, 3])) < 1e-3

    wl = W.config2(blocks=[0, 1000, 2000, 3599])
    acq = pt.make_acq_config(M=4096, spacing=5952, f_rel=0.0, f_bins=2.0, fdot_bins=2.0, a_rel=0.2)
    r = pt.pt_acquire(_cuda(wl.x), wl.fs, 5, acq)
    cfg = pt.make_config(D=5, NP=128, generations=1000, F=0.5, CR=0.9, seed=3, t0=wl.t0)
    g = {k: v.cpu().numpy() for k, v in pt.pt_fit_blocks(_cuda(wl.x), wl.fs, r["lo"], r["hi"], cfg).items()}
    # reference: the oracle's fit inside the same acquired boxes (the truth-centred literal boxes pin a1 on a face here)
    ref = oracle.fit_blocks(wl.x, wl.fs, r["lo"].cpu().numpy(), r["hi"].cpu().numpy(), NP=128, generations=500, F=0.5,
                            CR=0.9, seed=3)
    assert np.max(np.abs(g["best_rss"] - ref["best_rss"]) / ref["best_rss"]) < 1e-4
    assert np.max(np.abs(_wrap(g["best"][:, 2] - ref["best"][:, 2]))) < 5e-3
    assert np.max(np.abs(g["best"][:, 3] - ref["best"][:, 3])) < 1e-3


def test_invalid_acquisition_arguments(pt):
    wl = W.config0(cases=[0])
    for kw in (dict(M=100, spacing=10), dict(M=512, spacing=300), dict(M=4, spacing=10), dict(M=16384, spacing=1),
               dict(M=256, spacing=100, f_rel=-1.0)):
        with pytest.raises(pt.PtError):
            pt.pt_acquire(_cuda(wl.x), wl.fs, 5, pt.make_acq_config(**kw))


def test_track_auto_host_is_the_composition_of_the_device_calls(pt):
    """pt_track_auto_host (PAPER.md:250-252 process flow on host buffers: acquisition -> fit -> continuity check and
    re-search -> products) gives bit-identical results to the four device entry points called in turn."""
    wl = W.config1(blocks=range(10), generations=150, NP=40)
    x = wl.x.copy()
    x[6] = (wl.sigma * np.random.default_rng(3).standard_normal(wl.N)).astype(np.float32)     # the carrier drops out
    M = 2048
    acq = pt.make_acq_config(M=M, spacing=(wl.N - M) // 2, f_rel=0.0, f_bins=2.0, fdot_bins=2.0, a_rel=0.2)
    retry = pt.make_retry_config(phi_tol=0.5, F_tol=0.5, f_floor=2.0, fdot_floor=2.0)
    cfg = pt.make_config(D=5, NP=40, generations=150, seed=8, t0=wl.t0)
    h = pt.pt_track_auto_host(torch.from_numpy(x), wl.fs, cfg, acq, retry, 0.0, [2, 5])
    xd = _cuda(x)
    r = pt.pt_acquire(xd, wl.fs, 5, acq)
    fit = pt.pt_fit_blocks(xd, wl.fs, r["lo"], r["hi"], cfg)
    att = pt.pt_refit_doubtful(xd, wl.fs, r["lo"], r["hi"], cfg, retry, fit)
    per_block, total, ivs = pt.pt_doppler_products(fit["best"], wl.T, 0.0, [2, 5])
    assert np.array_equal(h["best"].numpy(), fit["best"].cpu().numpy())
    assert np.array_equal(h["status"].numpy(), fit["status"].cpu().numpy())
    assert np.array_equal(h["attempts"].numpy(), att.cpu().numpy())
    assert np.array_equal(h["lo"].numpy(), r["lo"].cpu().numpy()) and np.array_equal(h["hi"].numpy(), r["hi"].cpu().numpy())
    assert np.array_equal(h["total_phase"].numpy(), total.cpu().numpy())
    assert np.array_equal(h["intervals"][1].numpy(), ivs[1].cpu().numpy())
    # the dropped block is searched again (abandonment itself is covered by test_gpu_retry: here one of its borders may
    # pass the check by chance); the rest of the track is solved without caller ranges
    a = h["attempts"].numpy()
    assert a[6] >= 1
    ok = [b for b in range(10) if b != 6]
    assert np.all((h["status"].numpy()[ok] & 4) == 0)
    assert np.max(np.abs(h["best"].numpy()[ok, 3] - wl.truth[ok, 3])) < 0.02
    # without retry the same call stops after the fit
    h2 = pt.pt_track_auto_host(torch.from_numpy(x), wl.fs, cfg, acq, None, 0.0, [])
    assert int(h2["attempts"].sum()) == 0
