"""GPU parity of row f-1, second part: continuity check, run-time ranges and re-search of doubtful
blocks (reading R25) -- pt_refit_doubtful against the oracle's
refit_doubtful on the same scenarios.  The flag decisions compare residuals of fitted parameters with thresholds, so the
scenarios keep a clear margin (wrong ranges miss the true frequency by > 8 Hz; a block without carrier): the sets of
doubtful blocks, the attempt counts and the abandoned bit must be identical, re-fitted parameters within the usual bars.
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


def _run(pt, wl, x, lo, hi, *, NP, G, seed, retry_kw):
    cfg = pt.make_config(D=wl.D, NP=NP, generations=G, F=0.5, CR=0.9, seed=seed, t0=wl.t0)
    xd, lod, hid = _cuda(x), _cuda(lo), _cuda(hi)
    fit = pt.pt_fit_blocks(xd, wl.fs, lod, hid, cfg)
    first = {k: v.cpu().numpy().copy() for k, v in fit.items()}
    attempts = pt.pt_refit_doubtful(xd, wl.fs, lod, hid, cfg, pt.make_retry_config(**retry_kw), fit)
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in fit.items()}
    g.update(attempts=attempts.cpu().numpy(), lo=lod.cpu().numpy(), hi=hid.cpu().numpy())
    of = oracle.fit_blocks(x, wl.fs, lo, hi, NP=NP, generations=G, seed=seed)
    o = oracle.refit_doubtful(x, wl.fs, lo, hi, of["best"], of["best_rss"], of["status"], NP=NP, generations=G, seed=seed,
                              **retry_kw)
    return first, g, o


def test_wrong_ranges_are_found_and_repaired(pt):
    wl = W.config1(blocks=range(8), generations=150, NP=40)
    lo, hi = wl.lo.copy(), wl.hi.copy()
    for b in (2, 5):
        lo[b, 3] = wl.truth[b, 3] + 8.0
        hi[b, 3] = wl.truth[b, 3] + 30.0
    kw = dict(phi_tol=0.5, F_tol=0.5, f_floor=2.0, fdot_floor=2.0)
    first, g, o = _run(pt, wl, wl.x, lo, hi, NP=40, G=150, seed=5, retry_kw=kw)
    assert list(g["attempts"]) == list(o["attempts"]) == [0, 0, 1, 0, 0, 1, 0, 0]
    assert np.array_equal(g["status"] & 4, o["status"] & 4) and not np.any(g["status"] & 4)
    keep = [0, 1, 3, 4, 6, 7]
    assert np.array_equal(g["best"][keep], first["best"][keep])                  # trusted blocks are untouched
    assert np.max(np.abs(_wrap(g["best"][:, 2] - o["best"][:, 2]))) < 5e-3
    assert np.max(np.abs(g["best"][:, 3] - o["best"][:, 3])) < 1e-3
    assert np.max(np.abs(g["best_rss"] - o["best_rss"]) / o["best_rss"]) < 1e-4
    # the new ranges: same formulas from neighbours that agree to ~1e-4 Hz
    assert np.max(np.abs(g["lo"] - o["lo"])) < 1e-2 and np.max(np.abs(g["hi"] - o["hi"])) < 1e-2
    assert np.array_equal(g["lo"][keep], lo[keep]) and np.array_equal(g["hi"][keep], hi[keep])
    assert np.all(g["lo"][[2, 5], 3] <= wl.truth[[2, 5], 3]) and np.all(wl.truth[[2, 5], 3] <= g["hi"][[2, 5], 3])
    assert np.array_equal(g["lo"][[2, 5], 2], [-np.pi, -np.pi])


def test_block_without_carrier_is_abandoned(pt):
    wl = W.config1(blocks=range(6), generations=100, NP=30)
    x = wl.x.copy()
    x[3] = (wl.sigma * np.random.default_rng(1).standard_normal(wl.N)).astype(np.float32)
    kw = dict(phi_tol=0.3, F_tol=0.2, f_floor=2.0, fdot_floor=2.0)
    first, g, o = _run(pt, wl, x, wl.lo, wl.hi, NP=30, G=100, seed=2, retry_kw=kw)
    assert list(g["attempts"]) == list(o["attempts"]) == [0, 0, 0, 3, 0, 0]
    assert list(g["status"] & 4) == list(o["status"] & 4) == [0, 0, 0, 4, 0, 0]
    assert abs((g["hi"][3, 3] - g["lo"][3, 3]) - (o["hi"][3, 3] - o["lo"][3, 3])) < 1e-2


def test_nothing_to_do_and_many_blocks(pt):
    """A clean track: no block is touched.  Then 300 blocks (two waves of the persistent grid) with every 37th range
    wrong: the re-search runs on the selected blocks only and repairs all of them."""
    wl = W.config2(blocks=range(300), generations=120, NP=32)
    cfg = pt.make_config(D=5, NP=32, generations=120, seed=9, t0=wl.t0)
    xd = _cuda(wl.x)
    lo, hi = wl.lo.copy(), wl.hi.copy()
    lod, hid = _cuda(lo), _cuda(hi)
    fit = pt.pt_fit_blocks(xd, wl.fs, lod, hid, cfg)
    retry = pt.make_retry_config(phi_tol=1.0, F_tol=1.0, f_floor=2.0, fdot_floor=2.0)
    before = fit["best"].clone()
    att = pt.pt_refit_doubtful(xd, wl.fs, lod, hid, cfg, retry, fit)
    assert int(att.sum()) == 0 and torch.equal(before, fit["best"])
    bad = list(range(5, 300, 37))
    for b in bad:
        lo[b, 3] = wl.truth[b, 3] + 20.0
        hi[b, 3] = wl.truth[b, 3] + 60.0
    lod, hid = _cuda(lo), _cuda(hi)
    fit2 = pt.pt_fit_blocks(xd, wl.fs, lod, hid, cfg)
    att = pt.pt_refit_doubtful(xd, wl.fs, lod, hid, cfg, retry, fit2).cpu().numpy()
    assert sorted(np.nonzero(att)[0]) == bad and np.all(att[bad] == 1)
    assert not np.any(fit2["status"].cpu().numpy() & 4)
    d = (fit2["best"] - before).cpu().numpy()
    # 0 dB blocks and only 120 generations of 32 members: the two searches of a block end within the noise of each other
    # (Cramer-Rao sigma of config 2: 4.4e-3 Hz, 12 mrad), not at the converged-fit bars
    assert np.max(np.abs(d[:, 3])) < 2e-2 and np.max(np.abs(_wrap(d[:, 2]))) < 5e-2


def test_invalid_retry_arguments(pt):
    wl = W.config1(blocks=range(3), generations=5, NP=16)
    cfg = pt.make_config(D=5, NP=16, generations=5, t0=wl.t0)
    xd, lod, hid = _cuda(wl.x), _cuda(wl.lo), _cuda(wl.hi)
    fit = pt.pt_fit_blocks(xd, wl.fs, lod, hid, cfg)
    for kw in (dict(phi_tol=0.0, F_tol=1.0), dict(phi_tol=1.0, F_tol=1.0, grow=0.5), dict(phi_tol=1.0, F_tol=1.0, max_attempts=-1)):
        with pytest.raises(pt.PtError):
            pt.pt_refit_doubtful(xd, wl.fs, lod, hid, cfg, pt.make_retry_config(**kw), fit)


def test_re_search_over_a_selection_larger_than_one_wave(pt):
    """320 doubtful blocks of 960: the selection list is longer than one wave of the persistent grid (2 CTAs per SM), each work
    item writing to its own block's rows."""
    NB = 960
    wl = W.config2(blocks=range(NB), generations=120, NP=32)
    cfg = pt.make_config(D=5, NP=32, generations=120, seed=4, t0=wl.t0)
    xd = _cuda(wl.x)
    ref = pt.pt_fit_blocks(xd, wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg)["best"].cpu().numpy()
    lo, hi = wl.lo.copy(), wl.hi.copy()
    bad = list(range(1, NB, 3))
    for b in bad:
        lo[b, 3] = wl.truth[b, 3] + 20.0
        hi[b, 3] = wl.truth[b, 3] + 60.0
    lod, hid = _cuda(lo), _cuda(hi)
    fit = pt.pt_fit_blocks(xd, wl.fs, lod, hid, cfg)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    assert len(bad) > sms * pt.pt_fit_blocks_plan(NB, wl.N, cfg)["ctas_per_sm"]
    att = pt.pt_refit_doubtful(xd, wl.fs, lod, hid, cfg, pt.make_retry_config(phi_tol=1.0, F_tol=1.0, f_floor=2.0, fdot_floor=2.0),
                               fit).cpu().numpy()
    searched = set(int(b) for b in np.nonzero(att)[0])
    # every block with wrong ranges is searched again, once; so are the two end blocks (their only border is bad and
    # they cannot be told apart from their neighbour) and the odd pair of good blocks whose own common border failed the
    # check in the short 120-generation first fit
    assert set(bad) <= searched and {0, NB - 1} <= searched and len(searched - set(bad)) <= 16
    assert np.all(att[bad] == 1) and att.max() == 1
    assert not np.any(fit["status"].cpu().numpy() & 4)
    d = fit["best"].cpu().numpy() - ref
    good = [b for b in range(NB) if b not in searched]
    assert np.array_equal(d[good], np.zeros_like(d[good]))
    # 320 pairs of short searches: the bulk within the bars of the 160-block version of this test, the extremes within 10 sigma
    assert np.quantile(np.abs(d[bad, 3]), 0.99) < 2e-2 and np.quantile(np.abs(_wrap(d[bad, 2])), 0.99) < 5e-2
    assert np.max(np.abs(d[bad, 3])) < 4e-2 and np.max(np.abs(_wrap(d[bad, 2]))) < 0.12
