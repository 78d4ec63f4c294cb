"""GPU robustness cases of the DE kernel (through the C ABI): non-finite samples and inverted boxes are flagged per block in the
status word and never disturb the other blocks of the launch (an all-NaN objective used to index out of the
population; include/pt.h status bits 3 and 4)."""
import ctypes as C

import numpy as np
import pytest

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


def _fit(pt, x, wl, lo=None, hi=None, strategy=1, NP=60, G=60, seed=5):
    cfg = pt.make_config(D=5, NP=NP, generations=G, seed=seed, t0=wl.t0, strategy=strategy)
    r = pt.pt_fit_blocks(torch.from_numpy(np.ascontiguousarray(x)).cuda(), wl.fs,
                         torch.from_numpy(wl.lo if lo is None else lo).cuda(), torch.from_numpy(wl.hi if hi is None else hi).cuda(), cfg)
    torch.cuda.synchronize()          # a sticky fault (the old out-of-bounds read) would surface here
    return {k: v.cpu().numpy() for k, v in r.items()}


@pytest.mark.parametrize("strategy", [1, 2, 3])
@pytest.mark.parametrize("bad_value", [np.nan, np.inf, -np.inf])
def test_non_finite_sample_flags_its_block_only(pt, strategy, bad_value):
    """One NaN / Inf sample makes every member's objective of that block non-finite: the block gets status bit 3, the
    launch survives, and the other blocks' results are bit-identical to a launch without the bad sample.  Strategies 2 and 3
    index the population with the per-generation argmin, the path that used to run out of bounds."""
    wl = W.config0(cases=range(6))
    clean = _fit(pt, wl.x, wl, strategy=strategy)
    x = wl.x.copy()
    x[2, 417] = bad_value
    got = _fit(pt, x, wl, strategy=strategy)
    assert got["status"][2] & 8, got["status"]
    assert not np.isfinite(got["best_rss"][2])
    assert np.all(np.isfinite(got["best"][2])) and np.all(got["best"][2] >= wl.lo[2]) and np.all(got["best"][2] <= wl.hi[2])
    others = [0, 1, 3, 4, 5]
    assert np.all((got["status"][others] & 8) == 0)
    assert np.array_equal(got["best"][others], clean["best"][others])
    assert np.array_equal(got["best_rss"][others], clean["best_rss"][others])
    # the library is still usable afterwards (no sticky context error)
    again = _fit(pt, wl.x, wl, strategy=strategy)
    assert np.array_equal(again["best"], clean["best"])


def test_non_finite_sample_in_a_large_launch_cluster_and_streamed_paths(pt):
    """The same through the persistent loop (more blocks than CTAs) and the streamed path (N beyond shared memory)."""
    wl = W.single_tone_blocks(range(400), 512, 512.0, config=4, f_range=(20, 60))
    x = wl.x.copy()
    x[123, 5] = np.nan
    x[399, 511] = np.inf
    got = _fit(pt, x, wl, NP=16, G=8)
    bad = np.nonzero(got["status"] & 8)[0]
    assert list(bad) == [123, 399]
    wl2 = W.single_tone_blocks(range(3), 65536, 65536.0, config=4)
    x2 = wl2.x.copy()
    x2[1, 40000] = np.nan
    import os
    old = os.environ.get("PT_CLUSTER")
    os.environ["PT_CLUSTER"] = "1"          # test hook (include/pt.h): single-CTA plan -> the streamed path
    try:
        got2 = _fit(pt, x2, wl2, NP=32, G=3)
    finally:
        if old is None:
            os.environ.pop("PT_CLUSTER", None)
        else:
            os.environ["PT_CLUSTER"] = old
    assert list(np.nonzero(got2["status"] & 8)[0]) == [1]


def test_inverted_box_sets_status_bit4_on_the_device_path_and_is_an_error_on_the_host_path(pt):
    wl = W.config0(cases=range(4))
    lo, hi = wl.lo.copy(), wl.hi.copy()
    lo[1, 3], hi[1, 3] = hi[1, 3], lo[1, 3]          # block 1: lo > hi in the frequency coordinate
    lo[3, 0] = np.nan                                 # block 3: NaN bound
    got = _fit(pt, wl.x, wl, lo=lo, hi=hi)
    assert list(np.nonzero(got["status"] & 16)[0]) == [1, 3]
    clean = _fit(pt, wl.x, wl)
    assert np.array_equal(got["best"][[0, 2]], clean["best"][[0, 2]])
    # host entry point: checked synchronously
    cfg = pt.make_config(D=5, NP=60, generations=5, seed=5, t0=wl.t0)
    with pytest.raises(pt.PtError, match="lo > hi"):
        pt.pt_track_host(torch.from_numpy(wl.x), wl.fs, torch.from_numpy(lo), torch.from_numpy(hi), cfg)


def test_host_entry_point_cache_can_be_released_and_recreated(pt):
    """pt_track_host keeps a memory pool and a stream per device between calls (include/pt.h); releasing them must leave the
    library usable and the results unchanged."""
    wl = W.config0(cases=range(3))
    cfg = pt.make_config(D=5, NP=60, generations=40, seed=5, t0=wl.t0)
    args = (torch.from_numpy(wl.x), wl.fs, torch.from_numpy(wl.lo), torch.from_numpy(wl.hi), cfg, 0.0, [1])
    a = pt.pt_track_host(*args)
    b = pt.pt_track_host(*args)            # second call: served from the pool
    pt.pt_host_cache_release()
    pt.pt_host_cache_release()             # idempotent
    c = pt.pt_track_host(*args)
    for k in ("best", "best_rss", "status", "total_phase"):
        assert torch.equal(a[k], b[k]) and torch.equal(a[k], c[k]), k
