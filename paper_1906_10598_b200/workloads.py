"""Seeded synthetic open-loop tracking workloads (numpy only).

These are the input generators shared by the tests (oracle side and CUDA side) and ``bench.py``.
They stand in for the paper's Mars Express / Chang'E-4 baseband recordings (PAPER.md:51, :94,
Table 3 at :104-117), which are not available; shapes and signal structure follow
BASELINE.json's five configs and SURVEY.md section 8(d).  Nothing of the *method* (objective,
DE, Doppler products) lives here: this module only synthesises ``x = A(t) cos(phi(t)) + noise``
from an analytic Doppler profile, and states the truth and the parameter boxes that go with it.

Recipe:
  * phase phi(t) is the analytic integral of the frequency profile f(t), evaluated in fp64 at the
    absolute sample times t = (b N + n)/fs; samples are cast to fp32 last;
  * noise is white Gaussian with sigma^2 = (A_ref^2/2)/10^(SNR/10);
  * every block b has its own generator ``default_rng([1906105980 + 1000*config + case, b])`` so
    that any subset of blocks can be produced without generating the whole track;
  * per-block truth theta = (a0, a1, phi0, f, fdot[, fddot]) is the profile evaluated at the block
    centre t_c = (b + 1/2) T, phi0 wrapped to (-pi, pi];
  * boxes: "literal" = theta -+ 0.2 |theta| for every coordinate (BASELINE.json config 0),
    "paper" = phi0 in [-pi, pi], a1 in -+0.2 a0/T, a0 and f -+20 %, fdot half-width
    max(0.2 |fdot|, 2/T^2), fddot half-width 150/pi.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 1906105980
PARAM_NAMES = ("a0", "a1", "phi0", "f", "fdot", "fddot")


@dataclass
class Workload:
    name: str
    config: int
    x: np.ndarray            # [B][N] float32 baseband samples
    fs: float                # sample rate [Hz]
    truth: np.ndarray        # [B][D] float64, profile at the block centres
    lo: np.ndarray           # [B][D] float64 box
    hi: np.ndarray           # [B][D] float64 box
    sigma: float             # noise standard deviation (of the reference amplitude)
    de: dict                 # NP, D, generations, F, CR
    block_index: np.ndarray  # [B] uint32 index of each block within the full track
    meta: dict = field(default_factory=dict)

    @property
    def B(self) -> int:
        return int(self.x.shape[0])

    @property
    def N(self) -> int:
        return int(self.x.shape[1])

    @property
    def T(self) -> float:
        return self.N / self.fs

    @property
    def D(self) -> int:
        return int(self.de["D"])

    @property
    def t0(self) -> float:
        return -self.N / (2.0 * self.fs)


def wrap_pi(v):
    """Wrap to (-pi, pi]."""
    return -((-np.asarray(v, dtype=np.float64) + np.pi) % (2.0 * np.pi) - np.pi)


def make_box(truth: np.ndarray, T: float, style: str = "literal"):
    truth = np.asarray(truth, dtype=np.float64)
    D = truth.shape[-1]
    if style == "literal":
        half = 0.2 * np.abs(truth)
        return truth - half, truth + half
    if style != "paper":
        raise ValueError("box style must be 'literal' or 'paper'")
    lo = np.empty_like(truth)
    hi = np.empty_like(truth)
    a0, f, fdot = truth[..., 0], truth[..., 3], truth[..., 4]
    lo[..., 0], hi[..., 0] = a0 - 0.2 * np.abs(a0), a0 + 0.2 * np.abs(a0)
    lo[..., 1], hi[..., 1] = -0.2 * np.abs(a0) / T, 0.2 * np.abs(a0) / T
    lo[..., 2], hi[..., 2] = -np.pi, np.pi
    lo[..., 3], hi[..., 3] = f - 0.2 * np.abs(f), f + 0.2 * np.abs(f)
    hw = np.maximum(0.2 * np.abs(fdot), 2.0 / T**2)
    lo[..., 4], hi[..., 4] = fdot - hw, fdot + hw
    if D == 6:
        hw3 = 150.0 / np.pi
        lo[..., 5], hi[..., 5] = truth[..., 5] - hw3, truth[..., 5] + hw3
    return lo, hi


def _block_times(b: int, N: int, fs: float) -> np.ndarray:
    n = np.arange(N, dtype=np.float64)
    return (float(b) * N + n) / fs


def _noise_sigma(a_ref: float, snr_db: float) -> float:
    return float(np.sqrt((a_ref**2 / 2.0) / 10.0 ** (snr_db / 10.0)))


# ------------------------------------------------------------------------------------------
# Configs 0 and 4: independent single-tone blocks, parameters drawn per block.
# ------------------------------------------------------------------------------------------
def single_tone_blocks(cases, N: int, fs: float, *, config: int, snr_db: float = 20.0, box: str = "literal",
                       noiseless: bool = False, de: dict | None = None, f_range=(50.0, 200.0),
                       a1_zero: bool = False) -> Workload:
    """Block k is drawn from ``default_rng([BASE_SEED + 1000*config + case_k, 0])`` as BASELINE.json config 0
    states: a0~U(0.5,1.5), a1~U(-0.1,0.1), phi0~U(-pi,pi), f~U(50,200) Hz, fdot~U(-1,1) Hz/s; the time axis
    is t in [-T/2, T/2) about the block centre.  ``a1_zero`` sets the amplitude slope to zero after the draw
    (the constant-amplitude signal of PAPER.md:153, Eq. 6; the other draws are unchanged)."""
    cases = list(cases)
    B = len(cases)
    T = N / fs
    t = -T / 2.0 + np.arange(N, dtype=np.float64) / fs
    x = np.empty((B, N), dtype=np.float32)
    truth = np.empty((B, 5), dtype=np.float64)
    sig = np.empty(B)
    for k, case in enumerate(cases):
        rng = np.random.default_rng([BASE_SEED + 1000 * config + int(case), 0])
        a0 = rng.uniform(0.5, 1.5)
        a1 = rng.uniform(-0.1, 0.1)
        if a1_zero:
            a1 = 0.0
        phi0 = rng.uniform(-np.pi, np.pi)
        f = rng.uniform(*f_range)
        fdot = rng.uniform(-1.0, 1.0)
        truth[k] = (a0, a1, phi0, f, fdot)
        sig[k] = _noise_sigma(a0, snr_db)
        s = (a0 + a1 * t) * np.cos(phi0 + 2.0 * np.pi * (f * t + fdot * t * t / 2.0))
        if not noiseless:
            s = s + sig[k] * rng.standard_normal(N)
        x[k] = s.astype(np.float32)
    lo, hi = make_box(truth, T, box)
    de = dict(de or dict(NP=60, D=5, generations=500, F=0.5, CR=0.9))
    return Workload(name="config%d" % config, config=config, x=x, fs=float(fs), truth=truth, lo=lo, hi=hi,
                    sigma=float(np.mean(sig)), de=de, block_index=np.arange(B, dtype=np.uint32),
                    meta={"cases": cases, "sigma_per_block": sig, "box": box, "noiseless": noiseless})


def config0(cases=(0,), **kw) -> Workload:
    """BASELINE.json config 0: one (or several independent) 1 s block(s) at fs = 1 kHz, SNR 20 dB."""
    return single_tone_blocks(cases, 1000, 1000.0, config=0, **kw)


def config4(N: int, NP: int, B: int = 1024, generations: int = 200, **kw) -> Workload:
    """BASELINE.json config 4 point: B blocks of N samples (fs = N Hz, T = 1 s), drawn as config 0."""
    de = dict(NP=NP, D=5, generations=generations, F=0.5, CR=0.9)
    wl = single_tone_blocks(range(B), N, float(N), config=4, de=de, **kw)
    wl.name = "config4_N%d_NP%d" % (N, NP)
    return wl


# ------------------------------------------------------------------------------------------
# Configs 1-3: one continuous track cut into contiguous blocks.
# ------------------------------------------------------------------------------------------
class _Profile:
    """Analytic frequency profile f(t), its integral (cycles), derivatives, and amplitude A(t)."""

    D = 5

    def cycles(self, t):  # integral of f from 0 to t
        raise NotImplementedError

    def f(self, t):
        raise NotImplementedError

    def fdot(self, t):
        raise NotImplementedError

    def fddot(self, t):
        raise NotImplementedError

    def amp(self, t):
        return np.ones_like(np.asarray(t, dtype=np.float64))

    def damp(self, t):
        return np.zeros_like(np.asarray(t, dtype=np.float64))


class _Cubic(_Profile):  # config 1: f = 1000 + 5 t + 0.02 t^2 + 1e-4 t^3
    def cycles(self, t):
        return 1000.0 * t + 2.5 * t**2 + (0.02 / 3.0) * t**3 + 2.5e-5 * t**4

    def f(self, t):
        return 1000.0 + 5.0 * t + 0.02 * t**2 + 1e-4 * t**3

    def fdot(self, t):
        return 5.0 + 0.04 * t + 3e-4 * t**2

    def fddot(self, t):
        return 0.04 + 6e-4 * t


class _Track(_Profile):  # config 2: f = 2000 + 30 sin(2 pi t/3600) + 1e-4 t^2, A = 1 + 0.05 sin(2 pi t/600)
    w = 2.0 * np.pi / 3600.0
    wa = 2.0 * np.pi / 600.0

    def cycles(self, t):
        return 2000.0 * t + (30.0 / self.w) * (1.0 - np.cos(self.w * t)) + (1e-4 / 3.0) * t**3

    def f(self, t):
        return 2000.0 + 30.0 * np.sin(self.w * t) + 1e-4 * t**2

    def fdot(self, t):
        return 30.0 * self.w * np.cos(self.w * t) + 2e-4 * t

    def fddot(self, t):
        return -30.0 * self.w**2 * np.sin(self.w * t) + 2e-4

    def amp(self, t):
        return 1.0 + 0.05 * np.sin(self.wa * t)

    def damp(self, t):
        return 0.05 * self.wa * np.cos(self.wa * t)


class _Occultation(_Profile):  # config 3: f = 5000 + 200 tanh((t-1800)/60), amplitude fade
    D = 6

    def cycles(self, t):
        u = (np.asarray(t, dtype=np.float64) - 1800.0) / 60.0
        lc = np.logaddexp(u, -u) - np.log(2.0)            # ln cosh(u), overflow-free
        lc0 = np.logaddexp(-30.0, 30.0) - np.log(2.0)
        return 5000.0 * t + 200.0 * 60.0 * (lc - lc0)

    def f(self, t):
        return 5000.0 + 200.0 * np.tanh((t - 1800.0) / 60.0)

    def fdot(self, t):
        return (200.0 / 60.0) / np.cosh((t - 1800.0) / 60.0) ** 2

    def fddot(self, t):
        u = (t - 1800.0) / 60.0
        return -2.0 * (200.0 / 3600.0) * np.tanh(u) / np.cosh(u) ** 2

    def amp(self, t):
        d = np.asarray(t, dtype=np.float64) - 1800.0
        fade = 1.0 - 0.9 * 0.5 * (1.0 + np.cos(np.pi * d / 120.0))
        return np.where(np.abs(d) < 120.0, fade, 1.0)

    def damp(self, t):
        d = np.asarray(t, dtype=np.float64) - 1800.0
        dv = 0.9 * 0.5 * (np.pi / 120.0) * np.sin(np.pi * d / 120.0)
        return np.where(np.abs(d) < 120.0, dv, 0.0)


def _track(config: int, prof: _Profile, B_full: int, N: int, fs: float, snr_db: float, de: dict, blocks, case: int,
           box: str, noiseless: bool) -> Workload:
    T = N / fs
    blocks = np.arange(B_full) if blocks is None else np.asarray(list(blocks), dtype=np.int64)
    B = len(blocks)
    D = prof.D
    sigma = _noise_sigma(1.0, snr_db)
    x = np.empty((B, N), dtype=np.float32)
    for k, b in enumerate(blocks):
        t = _block_times(int(b), N, fs)
        s = prof.amp(t) * np.cos(2.0 * np.pi * prof.cycles(t))
        if not noiseless:
            rng = np.random.default_rng([BASE_SEED + 1000 * config + case, int(b)])
            s = s + sigma * rng.standard_normal(N)
        x[k] = s.astype(np.float32)
    tc = (blocks.astype(np.float64) + 0.5) * T
    truth = np.empty((B, D), dtype=np.float64)
    truth[:, 0] = prof.amp(tc)
    truth[:, 1] = prof.damp(tc)
    truth[:, 2] = wrap_pi(2.0 * np.pi * np.fmod(prof.cycles(tc), 1.0))
    truth[:, 3] = prof.f(tc)
    truth[:, 4] = prof.fdot(tc)
    if D == 6:
        truth[:, 5] = prof.fddot(tc)
    lo, hi = make_box(truth, T, box)
    edges_l = blocks.astype(np.float64) * T
    dphi_true = 2.0 * np.pi * (prof.cycles(edges_l + T) - prof.cycles(edges_l))   # exact phase advance per block
    return Workload(name="config%d" % config, config=config, x=x, fs=float(fs), truth=truth, lo=lo, hi=hi,
                    sigma=sigma, de=dict(de), block_index=blocks.astype(np.uint32),
                    meta={"case": case, "box": box, "noiseless": noiseless, "B_full": B_full, "tc": tc,
                          "dphi_true": dphi_true, "fddot_true": prof.fddot(tc)})


def config1(blocks=None, case: int = 0, box: str = "literal", noiseless: bool = False, **de_over) -> Workload:
    """60 contiguous 1 s blocks at 10 kHz from f(t) = 1000 + 5t + 0.02t^2 + 1e-4t^3 Hz, A = 1, SNR 10 dB."""
    de = dict(NP=100, D=5, generations=1000, F=0.5, CR=0.9)
    de.update(de_over)
    return _track(1, _Cubic(), 60, 10000, 1e4, 10.0, de, blocks, case, box, noiseless)


def config2(blocks=None, case: int = 0, box: str = "literal", noiseless: bool = False, **de_over) -> Workload:
    """3600 contiguous 1 s blocks at 16 kHz, f(t) = 2000 + 30 sin(2 pi t/3600) + 1e-4 t^2 Hz, SNR 0 dB."""
    de = dict(NP=128, D=5, generations=1000, F=0.5, CR=0.9)
    de.update(de_over)
    return _track(2, _Track(), 3600, 16000, 16e3, 0.0, de, blocks, case, box, noiseless)


def config3(blocks=None, case: int = 0, box: str = "literal", noiseless: bool = False, **de_over) -> Workload:
    """36000 contiguous 0.1 s blocks at 100 kHz, f(t) = 5000 + 200 tanh((t-1800)/60) Hz, fade, SNR 10 dB, D = 6."""
    de = dict(NP=128, D=6, generations=1500, F=0.5, CR=0.9)
    de.update(de_over)
    return _track(3, _Occultation(), 36000, 10000, 1e5, 10.0, de, blocks, case, box, noiseless)


def oracle_subset(config: int) -> list[int]:
    """The blocks on which configs 2 and 3 are oracle-checked: one 60-block run plus a stride."""
    if config == 2:
        return sorted(set(range(60)) | set(range(0, 3600, 100)))
    if config == 3:
        return sorted(set(range(60)) | set(range(0, 36000, 1000)))
    raise ValueError("subset is defined for configs 2 and 3")


# ------------------------------------------------------------------------------------------
# Quantised recordings (Table 3: 8/16-bit narrow-band and 1/2/4/8-bit wide-band modes).
# This is the receiver's A/D converter, i.e. input synthesis; unpacking belongs to the method (oracle / CUDA path).
# ------------------------------------------------------------------------------------------
def quantise(x: np.ndarray, bits: int):
    """Quantise fp32 samples x[B][N] to `bits`-wide codes and pack them, fields from the least significant bit of
    each byte upwards (16-bit: little-endian).  Returns (xq uint8 [B][row_bytes], quant dict) with
    quant = dict(bits, is_signed, scale, offset) such that the sample value is scale * (code + offset).

    8 and 16 bits: two's complement, full scale = the largest |x| of the array.
    1, 2, 4 bits: offset binary with L = 2^bits levels at (code - (L-1)/2) * step; step = 2 rms (1 bit: levels
    +-rms), rms (2 bits: thresholds at 0 and +-rms, close to the optimal 4-level quantiser of Gaussian noise),
    0.335 rms (4 bits, the optimal 16-level step)."""
    x = np.asarray(x, dtype=np.float32)
    B, N = x.shape
    if bits in (8, 16):
        full = float(np.max(np.abs(x)))
        qmax = (1 << (bits - 1)) - 1
        scale = full / qmax if full > 0 else 1.0
        code = np.clip(np.rint(x.astype(np.float64) / scale), -qmax - 1, qmax).astype(np.int64)
        quant = dict(bits=bits, is_signed=True, scale=scale, offset=0.0)
        if bits == 8:
            xq = code.astype(np.int8).view(np.uint8)
        else:
            xq = code.astype("<i2").view(np.uint8).reshape(B, 2 * N)
        return np.ascontiguousarray(xq), quant
    if bits not in (1, 2, 4):
        raise ValueError("bits must be 1, 2, 4, 8 or 16")
    if (N * bits) % 8:
        raise ValueError("N * bits must be a multiple of 8")
    L = 1 << bits
    rms = float(np.sqrt(np.mean(x.astype(np.float64) ** 2)))
    step = {1: 2.0, 2: 1.0, 4: 0.335}[bits] * rms
    offset = -(L - 1) / 2.0
    code = np.clip(np.floor(x.astype(np.float64) / step - offset + 0.5), 0, L - 1).astype(np.uint8)
    per = 8 // bits
    fields = code.reshape(B, N // per, per).astype(np.uint16)
    shifts = (np.arange(per) * bits).astype(np.uint16)
    xq = np.bitwise_or.reduce(fields << shifts, axis=-1).astype(np.uint8)
    return np.ascontiguousarray(xq), dict(bits=bits, is_signed=False, scale=step, offset=offset)


# ------------------------------------------------------------------------------------------
# Paper-shaped blocks (PAPER.md:51 footnote 2 "the data block is usually 2 seconds and sampling is 200KHz"; :94 "the
# data block size is about 400K ... evaluated by the DE solver ~80,000 times"; Table 4: Dim_XC 6, itermax 200, F_XC 0.5,
# CR_XC 0.85, strategy 3).  NP = 400 = 80,000 / 200.  Stand-in for the Mars Express recording the paper times.
# ------------------------------------------------------------------------------------------
def paper_blocks(B: int = 148, case: int = 0, N: int = 400000, fs: float = 200000.0, snr_db: float = -13.0) -> Workload:
    """B independent 2 s blocks of 400 000 samples at 200 kHz: a0~U(0.8,1.2), a1~U(-0.02,0.02), phi0~U(-pi,pi),
    f~U(20,80) kHz, fdot~U(-30,30) Hz/s, fddot~U(-0.5,0.5) Hz/s^2; -13 dB per sample = 40 dB-Hz.  Boxes are of the
    run-time (tracking) kind: phi0 a full turn, f +-2/T, fdot +-4/T^2, fddot +-16/T^3 about the
    truth, a0 +-10 %, a1 +-0.2 a0/T."""
    T = N / fs
    t = -T / 2.0 + np.arange(N, dtype=np.float64) / fs
    x = np.empty((B, N), dtype=np.float32)
    truth = np.empty((B, 6), dtype=np.float64)
    sig = np.empty(B)
    for k in range(B):
        rng = np.random.default_rng([BASE_SEED + 5000 + int(case), k])
        a0, a1 = rng.uniform(0.8, 1.2), rng.uniform(-0.02, 0.02)
        phi0, f = rng.uniform(-np.pi, np.pi), rng.uniform(20e3, 80e3)
        fdot, fddot = rng.uniform(-30.0, 30.0), rng.uniform(-0.5, 0.5)
        truth[k] = (a0, a1, phi0, f, fdot, fddot)
        sig[k] = _noise_sigma(a0, snr_db)
        ph = phi0 + 2.0 * np.pi * (f * t + fdot * t * t / 2.0 + fddot * t**3 / 6.0)
        x[k] = ((a0 + a1 * t) * np.cos(ph) + sig[k] * rng.standard_normal(N)).astype(np.float32)
    lo, hi = truth.copy(), truth.copy()
    hw = np.array([0.0, 0.0, 0.0, 2.0 / T, 4.0 / T**2, 16.0 / T**3])
    lo -= hw; hi += hw
    lo[:, 0], hi[:, 0] = 0.9 * truth[:, 0], 1.1 * truth[:, 0]
    lo[:, 1], hi[:, 1] = -0.2 * truth[:, 0] / T, 0.2 * truth[:, 0] / T
    lo[:, 2], hi[:, 2] = -np.pi, np.pi
    de = dict(NP=400, D=6, generations=200, F=0.5, CR=0.85, strategy=3)
    return Workload(name="paper_blocks", config=5, x=x, fs=float(fs), truth=truth, lo=lo, hi=hi, sigma=float(np.mean(sig)),
                    de=de, block_index=np.arange(B, dtype=np.uint32), meta={"sigma_per_block": sig, "box": "tracking"})
