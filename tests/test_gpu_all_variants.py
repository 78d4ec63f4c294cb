"""Every kernel variant once, on small inputs, with a device synchronisation after each: the launch geometries and shared-memory
layouts of all plans (this is the run that stands in for compute-sanitizer, which is closed on the GPU pool: profiles/r2_sanitizers.md).
A bad layout or a missed barrier phase shows up here as a CUDA error or a hang, not as a wrong number."""
import os

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


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _fit(pt, wl, NP, G, D=5, strategy=1, objective=0, env=None, quant=None):
    old = {}
    for k, v in (env or {}).items():
        old[k] = os.environ.get(k)
        os.environ[k] = v
    try:
        cfg = pt.make_config(D=D, NP=NP, generations=G, seed=3, t0=wl.t0, strategy=strategy, objective=objective)
        plan = pt.pt_fit_blocks_plan(wl.B, wl.N, cfg)
        lo, hi = wl.lo.copy(), wl.hi.copy()
        if objective:
            lo[:, 0] = hi[:, 0] = wl.truth[:, 0]
            lo[:, 1] = hi[:, 1] = 0.0
        if quant:
            xq, qd = W.quantise(wl.x, quant)
            q = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
            r = pt.pt_fit_blocks(_cuda(xq), wl.fs, _cuda(lo), _cuda(hi), cfg, quant=q, N=wl.N)
        else:
            r = pt.pt_fit_blocks(_cuda(wl.x), wl.fs, _cuda(lo), _cuda(hi), cfg, want_pop=True)
        torch.cuda.synchronize()
        return plan, {k: v.cpu().numpy() for k, v in r.items()}
    finally:
        for k, v in old.items():
            if v is None:
                os.environ.pop(k, None)
            else:
                os.environ[k] = v


SMALL = lambda: W.single_tone_blocks(range(6), 1024, 1024.0, config=4, f_range=(20, 60))
CUBIC = lambda: W.single_tone_blocks(range(3), 1024, 1024.0, config=4, f_range=(20, 60))     # fs = 1 kHz: the cubic term matters inside a run
CASES = {
    # ---- pt_run_kernel (the automatic choice) ----
    "run resident D5, automatic clusters": (SMALL, dict(NP=16, G=3), dict(threads=1024, cluster=lambda k: k >= 2)),
    "run resident D5, single CTA": (SMALL, dict(NP=16, G=3, env={"PT_CLUSTER": "1"}), dict(threads=1024, cluster=1)),
    "run cluster of 8": (lambda: W.single_tone_blocks(range(2), 4096, 4096.0, config=4), dict(NP=16, G=2, env={"PT_CLUSTER": "8"}), dict(threads=1024, cluster=8)),
    "run cluster of 3, N % 4 == 2": (lambda: W.single_tone_blocks(range(2), 4098, 4098.0, config=4), dict(NP=16, G=2, env={"PT_CLUSTER": "3"}), dict(cluster=3)),
    "run strategy 3 + correlation": (SMALL, dict(NP=16, G=3, strategy=3, objective=1, env={"PT_CLUSTER": "1"}), dict(cluster=1)),
    "run resident D6 (cubic folded into the run's second derivative)": (lambda: W.config3(blocks=[10, 11, 12]), dict(NP=16, G=2, D=6, env={"PT_CLUSTER": "1"}), dict(threads=1024)),
    "run more members than threads": (SMALL, dict(NP=1024, G=1, env={"PT_CLUSTER": "1"}), dict(threads=1024)),
    "run 8 CTAs per SM (short blocks), one partly filled round": (lambda: W.single_tone_blocks(range(600), 2048, 2048.0, config=4, f_range=(20, 60)),
                                                                  dict(NP=16, G=2), dict(threads=128, ctas_per_sm=8)),
    "run 4 CTAs per SM + cluster tail": (lambda: W.single_tone_blocks(range(600), 2048, 2048.0, config=4, f_range=(20, 60)),
                                         dict(NP=272, G=2), dict(threads=256, ctas_per_sm=4, tail_cluster=lambda k: k >= 2)),
    "run 2 CTAs per SM": (lambda: W.single_tone_blocks(range(160), 512, 512.0, config=4, f_range=(20, 60)), dict(NP=8, G=2), dict(threads=512, ctas_per_sm=2)),
    "run streamed ring": (lambda: W.single_tone_blocks(range(2), 65536, 65536.0, config=4), dict(NP=16, G=1, env={"PT_CLUSTER": "1"}), dict(resident=0, threads=1024)),
    "run streamed ring, quantised 4 bit": (lambda: W.single_tone_blocks(range(2), 65536, 65536.0, config=4), dict(NP=16, G=1, quant=4, env={"PT_CLUSTER": "1"}), dict(resident=0)),
    "run quantised 2 bit": (SMALL, dict(NP=16, G=2, quant=2, env={"PT_CLUSTER": "1"}), dict(threads=1024)),
    # ---- pt_block_kernel (PT_KERNEL=classic) ----
    "classic resident D5, automatic clusters": (SMALL, dict(NP=16, G=3, env={"PT_KERNEL": "classic"}), dict(threads=512, cluster=lambda k: k >= 2)),
    "classic resident D5, single CTA": (SMALL, dict(NP=16, G=3, env={"PT_CLUSTER": "1", "PT_KERNEL": "classic"}), dict(threads=512, cluster=1)),
    "classic cluster of 8": (lambda: W.single_tone_blocks(range(2), 4096, 4096.0, config=4), dict(NP=16, G=2, env={"PT_CLUSTER": "8", "PT_KERNEL": "classic"}), dict(threads=512, cluster=8)),
    "classic strategy 3 + correlation": (SMALL, dict(NP=16, G=3, strategy=3, objective=1, env={"PT_CLUSTER": "1", "PT_KERNEL": "classic"}), dict(cluster=1)),
    "classic resident D6": (lambda: W.config3(blocks=[10, 11, 12]), dict(NP=16, G=2, D=6, env={"PT_CLUSTER": "1", "PT_KERNEL": "classic"}), dict(threads=512)),
    "classic persistent loop + tail launch": (lambda: W.single_tone_blocks(range(158), 512, 512.0, config=4, f_range=(20, 60)),
                                              dict(NP=8, G=2, env={"PT_KERNEL": "classic"}), dict(resident=1)),
    "classic streamed ring": (lambda: W.single_tone_blocks(range(2), 65536, 65536.0, config=4), dict(NP=16, G=1, env={"PT_CLUSTER": "1", "PT_KERNEL": "classic"}), dict(resident=0, threads=512)),
    "classic quantised 2 bit": (SMALL, dict(NP=16, G=2, quant=2, env={"PT_CLUSTER": "1", "PT_KERNEL": "classic"}), dict(threads=512)),
    # ---- pt_tc_kernel (PT_KERNEL=tc) ----
    "tensor-core D6, one block per CTA": (lambda: W.config3(blocks=[10, 11, 12]), dict(NP=32, G=2, D=6, env={"PT_CLUSTER": "1", "PT_KERNEL": "tc"}), dict(threads=640)),
    "tensor-core D5, two blocks per CTA + cluster tail": (lambda: W.single_tone_blocks(range(310), 512, 512.0, config=4, f_range=(20, 60)),
                                                          dict(NP=16, G=2, env={"PT_KERNEL": "tc"}), dict(threads=640, tail_cluster=lambda k: k >= 2)),
    "tensor-core quantised 8 bit": (SMALL, dict(NP=16, G=2, quant=8, env={"PT_CLUSTER": "1", "PT_KERNEL": "tc"}), dict(threads=640)),
    "tensor-core correlation objective": (SMALL, dict(NP=16, G=2, objective=1, env={"PT_CLUSTER": "1", "PT_KERNEL": "tc"}), dict(threads=640)),
}


@pytest.mark.parametrize("name", list(CASES))
def test_variant_runs_clean(pt, name):
    make, kw, expect = CASES[name]
    wl = make()
    kw = dict(kw)
    plan, r = _fit(pt, wl, kw.pop("NP"), kw.pop("G"), **kw)
    for k, v in expect.items():
        assert v(plan[k]) if callable(v) else plan[k] == v, (name, k, plan)
    assert np.all(np.isfinite(r["best_rss"])) and np.all(np.isfinite(r["best"])), name
    if not kw.get("objective"):
        assert np.all(r["best"] >= wl.lo) and np.all(r["best"] <= wl.hi), name
    assert np.all((r["status"] & (8 | 16)) == 0), name


def test_the_small_entry_points_run_clean(pt):
    small = SMALL()
    pop = (small.lo[:, None, :] + (small.hi - small.lo)[:, None, :] * np.random.default_rng(0).uniform(size=(small.B, 16, 5))).astype(np.float32)
    f = pt.pt_fitness(_cuda(small.x), small.fs, _cuda(pop))
    trk = W.config2(blocks=range(12), generations=3)
    acq = pt.make_acq_config(M=1024, spacing=2048, f_rel=0.0, f_bins=2.0, fdot_bins=2.0, a_rel=0.2)
    a = pt.pt_acquire(_cuda(trk.x), trk.fs, 5, acq)
    cfg = pt.make_config(D=5, NP=16, generations=3, seed=1, t0=trk.t0)
    lo, hi = _cuda(trk.lo), _cuda(trk.hi)
    r = pt.pt_fit_blocks(_cuda(trk.x), trk.fs, lo, hi, cfg)
    att = pt.pt_refit_doubtful(_cuda(trk.x), trk.fs, lo, hi, cfg, pt.make_retry_config(phi_tol=1e-3, F_tol=1e-3, max_attempts=2), r)
    pb, tot, iv = pt.pt_doppler_products(r["best"], trk.T, 0.0, [1, 4])
    torch.cuda.synchronize()
    assert bool(torch.isfinite(f).all()) and bool(torch.isfinite(a["lo"]).all()) and bool(torch.isfinite(tot).all())
    assert att.cpu().numpy().max() == 2          # thresholds far below the noise: every block is re-searched twice
