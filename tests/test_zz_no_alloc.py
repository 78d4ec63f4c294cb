"""pt_refit_doubtful_static (include/pt.h, csrc/pt_noalloc.cu): the continuity check and re-search of doubtful blocks
 with its scratch in the library's static device array -- for callers that cannot call cudaMalloc.
It must give what pt_refit_doubtful gives on a caller workspace (same kernels, same seeds: the fitted parameters are compared at
the bars of the other GPU tests and are in fact identical), on two calls in a row: the second call finds the first call's contents in
the array and a different scenario must not see them.  Collected last on purpose (the suite runs with pytest -x).
"""
import ctypes as C

import numpy as np
import pytest

from paper_1906_10598_b200 import workloads as W

torch = pytest.importorskip("torch")

PHI0_TOL, F_TOL, FIT_REL_TOL = 5e-3, 1e-3, 1e-4


def _wrap(d):
    return (np.asarray(d) + np.pi) % (2 * np.pi) - np.pi


def test_static_scratch_limit_is_enforced_without_a_gpu():
    """Sizes beyond the static array are refused with a clear message before any CUDA call (so this runs on the CPU box too)."""
    from paper_1906_10598_b200 import pt
    L = pt.lib()
    cap = L.pt_static_scratch_bytes()
    assert cap == 4 * 1024 * 1024
    cfg = pt.make_config(D=5, NP=32, generations=5, t0=-0.5)
    ok = pt.make_retry_config(phi_tol=1.0, F_tol=1.0)
    dummy = C.c_void_p(256)
    assert L.pt_refit_doubtful_workspace_bytes(36000, 10000, C.byref(cfg)) <= cap          # BASELINE config 3 fits
    too_many = 60000
    assert L.pt_refit_doubtful_workspace_bytes(too_many, 1000, C.byref(cfg)) > cap
    rc = L.pt_refit_doubtful_static(dummy, too_many, 1000, 1000.0, dummy, dummy, None, C.byref(cfg), C.byref(ok), dummy, dummy,
                                    dummy, dummy, None)
    assert rc == -2
    msg = L.pt_last_error_string().decode()
    assert "static array holds" in msg and "pt_refit_doubtful" in msg
    # blocks streamed from global memory need workspace rows of their own: refused as well
    assert L.pt_refit_doubtful_static(dummy, 200, 400000, 200000.0, dummy, dummy, None, C.byref(cfg), C.byref(ok), dummy, dummy,
                                      dummy, dummy, None) == -2
    assert L.pt_refit_doubtful_static(None, 4, 1000, 1000.0, dummy, dummy, None, C.byref(cfg), C.byref(ok), dummy, dummy, dummy,
                                      dummy, None) == -1


def _scenario(k):
    """Two different tracks with wrong ranges on different blocks (and different sizes, so the second call uses fewer bytes of the
    array than the first left behind)."""
    if k == 0:
        wl = W.config1(blocks=range(12), generations=150, NP=40)
        bad = (2, 5, 9)
    else:
        wl = W.config1(blocks=range(20, 28), generations=150, NP=40)
        bad = (2, 5)
    lo, hi = wl.lo.copy(), wl.hi.copy()
    for b in bad:
        lo[b, 3] = wl.truth[b, 3] + 8.0
        hi[b, 3] = wl.truth[b, 3] + 30.0
    return wl, lo, hi, bad


@pytest.mark.gpu
def test_static_entry_matches_the_workspace_path_on_two_calls_in_a_row():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device; there is no CPU fallback")
    from paper_1906_10598_b200 import pt
    pt.lib()
    retry = pt.make_retry_config(phi_tol=0.5, F_tol=0.5, f_floor=2.0, fdot_floor=2.0)
    for call in range(2):
        wl, lo, hi, bad = _scenario(call)
        cfg = pt.make_config(D=wl.D, NP=40, generations=150, F=0.5, CR=0.9, seed=5 + call, t0=wl.t0)
        xd = torch.from_numpy(np.ascontiguousarray(wl.x)).cuda()
        res = {}
        for which in ("workspace", "static"):
            lod, hid = torch.from_numpy(lo.copy()).cuda(), torch.from_numpy(hi.copy()).cuda()
            fit = pt.pt_fit_blocks(xd, wl.fs, lod, hid, cfg)
            if which == "workspace":
                att = pt.pt_refit_doubtful(xd, wl.fs, lod, hid, cfg, retry, fit)
            else:
                att = torch.full((wl.B,), -7, dtype=torch.int32, device=xd.device)          # the caller's buffer, pre-filled
                before = torch.cuda.memory_allocated()
                pt.pt_refit_doubtful_static(xd, wl.fs, lod, hid, cfg, retry, fit, att)
                assert torch.cuda.memory_allocated() == before          # nothing came from torch's allocator either
            torch.cuda.synchronize()
            res[which] = dict(best=fit["best"].cpu().numpy(), rss=fit["best_rss"].cpu().numpy(), status=fit["status"].cpu().numpy(),
                              att=att.cpu().numpy(), lo=lod.cpu().numpy(), hi=hid.cpu().numpy())
        w, s = res["workspace"], res["static"]
        searched = set(int(b) for b in np.nonzero(w["att"])[0])
        assert set(bad) <= searched and len(searched) <= len(bad) + 1 and w["att"].max() == 1, (call, w["att"])       # the scenario does re-search
        assert np.array_equal(s["att"], w["att"]) and np.array_equal(s["status"], w["status"]), call
        assert np.max(np.abs(_wrap(s["best"][:, 2] - w["best"][:, 2]))) < PHI0_TOL
        assert np.max(np.abs(s["best"][:, 3] - w["best"][:, 3])) < F_TOL
        assert np.max(np.abs(s["rss"] - w["rss"]) / w["rss"]) < FIT_REL_TOL
        assert np.max(np.abs(s["lo"] - w["lo"])) < 1e-2 and np.max(np.abs(s["hi"] - w["hi"])) < 1e-2
        # same kernels, same Philox keys, same launch geometry: in fact bit for bit
        assert np.array_equal(s["best"], w["best"]) and np.array_equal(s["lo"], w["lo"]) and np.array_equal(s["hi"], w["hi"]), call
        assert np.all(np.abs(s["best"][:, 3] - wl.truth[:, 3]) < 0.05), call          # and the repaired blocks found the carrier
