"""GPU parity of row f-4: quantised sample input (Table 3; reading R23),
unpacked in-kernel while a block is staged.  Bars: the unpacked samples are bit-exact against the oracle; the fit on
packed samples is bit-identical to the fit of the same library on the unpacked fp32 samples (the unpacking is the only
difference) and within the usual bars of the oracle's fit.
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


@pytest.mark.parametrize("bits", [1, 2, 4, 8, 16])
def test_unpack_bit_exact(pt, bits):
    rng = np.random.default_rng(100 + bits)
    B, N = 5, 10000
    row_bytes = N * bits // 8 + 5
    xq = rng.integers(0, 256, size=(B, row_bytes), dtype=np.uint8)
    for signed in (False, True):
        scale, offset = 0.0123 * (bits + 1), -0.5 * ((1 << bits) - 1) if not signed else 0.25
        q = pt.make_quant(bits, signed, scale, offset)
        got = pt.pt_unpack_samples(_cuda(xq), N, q).cpu().numpy()
        ref = oracle.unpack_samples(xq, N, bits, signed, scale, offset)
        assert np.array_equal(got, ref)


def _fit(pt, wl, x_or_xq, *, quant=None, G, NP, seed=3, want_pop=True):
    cfg = pt.make_config(D=wl.D, NP=NP, generations=G, F=0.5, CR=0.9, seed=seed, t0=wl.t0)
    r = pt.pt_fit_blocks(_cuda(x_or_xq), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg, want_pop=want_pop, quant=quant, N=wl.N)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in r.items()}


@pytest.mark.parametrize("bits", [1, 2, 4, 8, 16])
def test_fit_on_packed_samples_equals_fit_on_unpacked_samples(pt, bits):
    wl = W.config0(cases=range(5))
    xq, qd = W.quantise(wl.x, bits)
    q = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
    x = oracle.unpack_samples(xq, wl.N, qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
    a = _fit(pt, wl, xq, quant=q, G=60, NP=32)
    b = _fit(pt, wl, x, G=60, NP=32)
    for k in ("best", "best_rss", "status", "final_pop", "final_fit"):
        assert np.array_equal(a[k], b[k]), k


@pytest.mark.parametrize("K", [1, 4])
def test_fit_8bit_against_the_oracle(pt, K):
    """Full fits on 8-bit samples (the receiver's narrow-band format), single CTA and split over a cluster (every CTA
    unpacks its own slice of the row)."""
    wl = W.config0(cases=range(6))
    xq, qd = W.quantise(wl.x, 8)
    q = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
    x = oracle.unpack_samples(xq, wl.N, qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
    with _forced_cluster(K):
        g = _fit(pt, wl, xq, quant=q, G=500, NP=60, want_pop=False)
    o = oracle.fit_blocks(x, wl.fs, wl.lo, wl.hi, NP=60, generations=500, F=0.5, CR=0.9, seed=3)
    assert np.max(np.abs(_wrap(g["best"][:, 2] - o["best"][:, 2]))) < 5e-3
    assert np.max(np.abs(g["best"][:, 3] - o["best"][:, 3])) < 1e-3
    assert np.max(np.abs(g["best_rss"] - o["best_rss"]) / o["best_rss"]) < 1e-4


def test_streamed_blocks_and_ragged_rows(pt):
    """Blocks larger than shared memory are unpacked into the workspace row; N not a multiple of 4 or of the chunk."""
    with _forced_cluster(1):
        wl = W.single_tone_blocks(range(2), 65536 + 136, 65536.0, config=4, f_range=(50.0, 200.0))
        cfg = pt.make_config(D=5, NP=16, generations=3, t0=wl.t0)
        assert pt.pt_fit_blocks_plan(wl.B, wl.N, cfg)["resident"] == 0
        for bits in (2, 8):
            xq, qd = W.quantise(wl.x, bits)
            q = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
            x = oracle.unpack_samples(xq, wl.N, qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
            a = _fit(pt, wl, xq, quant=q, G=3, NP=16)
            b = _fit(pt, wl, x, G=3, NP=16)
            for k in ("best", "best_rss", "final_pop", "final_fit"):
                assert np.array_equal(a[k], b[k]), (bits, k)
    wl = W.single_tone_blocks(range(3), 1002, 1002.0, config=4, f_range=(50.0, 200.0))
    xq, qd = W.quantise(wl.x, 16)
    q = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
    x = oracle.unpack_samples(xq, wl.N, 16, True, qd["scale"], qd["offset"])
    a = _fit(pt, wl, xq, quant=q, G=5, NP=12)
    o = oracle.fit_blocks(x, wl.fs, wl.lo, wl.hi, NP=12, generations=5, F=0.5, CR=0.9, seed=3, want_pop=True)
    assert (np.all(a["final_pop"] == o["final_pop"].astype(np.float32), axis=-1)).mean() > 0.95


def test_track_host_q_equals_the_device_path(pt):
    wl = W.config1(blocks=range(6), generations=40)
    xq, qd = W.quantise(wl.x, 8)
    q = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
    cfg = pt.make_config(D=5, NP=32, generations=40, seed=5, t0=wl.t0)
    h = pt.pt_track_host(torch.from_numpy(xq), wl.fs, torch.from_numpy(wl.lo), torch.from_numpy(wl.hi), cfg, 0.0, [2, 3],
                         quant=q, N=wl.N)
    d = pt.pt_fit_blocks(_cuda(xq), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg, quant=q, N=wl.N)
    per_block, total, ivs = pt.pt_doppler_products(d["best"], wl.T, 0.0, [2, 3])
    assert np.array_equal(h["best"].numpy(), d["best"].cpu().numpy())
    assert np.array_equal(h["total_phase"].numpy(), total.cpu().numpy())
    assert np.array_equal(h["intervals"][1].numpy(), ivs[1].cpu().numpy())


def test_invalid_quant_is_rejected(pt):
    wl = W.config0(cases=[0])
    xq, qd = W.quantise(wl.x, 8)
    cfg = pt.make_config(D=5, NP=16, generations=1, t0=wl.t0)
    with pytest.raises(pt.PtError):
        pt.pt_fit_blocks(_cuda(xq), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg, quant=pt.make_quant(3, True, 1.0), N=wl.N)
    with pytest.raises(pt.PtError):
        pt.pt_fit_blocks(_cuda(xq[:, :500]), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg, quant=pt.make_quant(8, True, 1.0), N=wl.N)
    with pytest.raises(pt.PtError):
        pt.pt_unpack_samples(_cuda(xq), wl.N, pt.make_quant(8, True, float("nan")))


def test_paper_shaped_blocks(pt):
    """PAPER.md:51, :94, Table 4: 400 000 samples (2 s at 200 kHz), D = 6, strategy 3, F 0.5, CR 0.85, 200 iterations,
    NP = 400 (80 000 evaluations), 16-bit samples (Table 3), streamed through shared memory.  In bench.py's launch
    configuration on 4 blocks: every result is valid (its RSS is the oracle's objective at its own parameters), the
    chi^2 sits at the noise floor, phi0 and f land within 4 Cramer-Rao sigma of the truth."""
    wl = W.paper_blocks(B=4)
    xq, qd = W.quantise(wl.x, 16)
    q = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
    de = wl.de
    cfg = pt.make_config(D=6, NP=de["NP"], generations=de["generations"], F=de["F"], CR=de["CR"], seed=1, t0=wl.t0,
                         strategy=de["strategy"])
    with _forced_cluster(1):
        assert pt.pt_fit_blocks_plan(148, wl.N, cfg)["resident"] == 0
        g = pt.pt_fit_blocks(_cuda(xq), wl.fs, _cuda(wl.lo), _cuda(wl.hi), cfg, quant=q, N=wl.N)
    g = {k: v.cpu().numpy() for k, v in g.items()}
    x = oracle.unpack_samples(xq, wl.N, 16, True, qd["scale"], qd["offset"])
    for k in range(wl.B):
        assert abs(g["best_rss"][k] - oracle.rss(x[k], wl.fs, g["best"][k])) < 1e-4 * g["best_rss"][k]
        s2 = wl.meta["sigma_per_block"][k] ** 2
        assert abs(g["best_rss"][k] - (wl.N - 6) * s2) < 5 * s2 * np.sqrt(2.0 * wl.N)
        # Cramer-Rao bounds from the Fisher matrix of Eq. 2 in white noise
        t = wl.t0 + np.arange(wl.N) / wl.fs
        th = wl.truth[k]
        ph = th[2] + 2 * np.pi * (th[3] * t + th[4] * t * t / 2 + th[5] * t**3 / 6)
        A, c, sn = th[0] + th[1] * t, np.cos(ph), np.sin(ph)
        J = np.array([c, t * c, -A * sn, -A * sn * 2 * np.pi * t, -A * sn * np.pi * t * t, -A * sn * np.pi * t**3 / 3])
        sd = np.sqrt(np.diag(np.linalg.inv(J @ J.T / s2)))
        assert abs(_wrap(g["best"][k, 2] - wl.truth[k, 2])) < 4 * sd[2] + 1e-3
        assert abs(g["best"][k, 3] - wl.truth[k, 3]) < 4 * sd[3]
