"""fp64 oracle of the initial range determination (section 3.1.1 items 1-6).

TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/pt_oracle.c's header): only tests/, smoke() and bench.py's
cpu_baseline legs may import it; it shares no code with paper_1906_10598_b200/.

The paper's procedure, per data block:
  1. c0 (phase at the block centre): range [0, 2 pi]
  2. c1 (frequency at the block centre): "FFT computation of a small piece of data extracted from block center",
     range +-10 % of c1
  3. c2 (half the second derivative of the phase): "central difference method through three equally spaced
     frequency values near block center", each "calculated as step 2"
  4. c3: range [-50, 50]
  5. c4 (amplitude): "determined by FFT algorithm done at step 2", range +-10 %
  6. c5 (amplitude slope): range [-0.2 c4/T, 0.2 c4/T]

What the paper leaves open and DESIGN.md reading R24 fixes (identically here and, independently written, in the CUDA
path): the piece length M (a power of two) and the spacing S of the three pieces (in samples) are parameters; piece k
(k = -1, 0, 1) is samples [N/2 + k S - M/2, N/2 + k S + M/2) of the block; it is weighted by the periodic Hann window
w_m = 0.5 - 0.5 cos(2 pi m / M); the frequency is that of the largest |X_k|^2 over 1 <= k <= M/2 - 1 (lowest k on ties)
refined by a parabola through the logarithms of the three powers around it,
    delta = 0.5 (ln P[k-1] - ln P[k+1]) / (ln P[k-1] - 2 ln P[k] + ln P[k+1]),   f = (k + delta) fs / M;
the amplitude is 4 |X_k| / M divided by the Hann main-lobe factor sinc(delta) / (1 - delta^2); fdot is the central
difference (f_{+1} - f_{-1}) / (2 S / fs).  The library FFT (numpy.fft.rfft, fp64) is the step the paper names.

Ranges in this build's units theta = (a0, a1, phi0, f, fdot[, fddot]) (c1 = 2 pi f, c2 = pi fdot, c3 = (pi/3) fddot):
    phi0 in [-pi, pi]                       (a full turn, item 1)
    f    in f_c -+ max(f_rel |f_c|, f_bins fs/M)                     (item 2: f_rel = 0.1, f_bins = 0)
    fdot in fdot_est -+ fdot_bins (fs/M) / (S/fs)                    (the paper gives no range for c2; one frequency
                                                                      bin of error across one spacing per fdot_bins)
    fddot in -+ fddot_hw                                             (item 4: 50 * 3/pi = 47.75 Hz/s^2)
    a0   in a_est (1 -+ a_rel)                                       (item 5: a_rel = 0.1)
    a1   in -+ a1_rel a_est / T                                      (item 6: a1_rel = 0.2)
"""
from __future__ import annotations

import numpy as np

DEFAULTS = dict(f_rel=0.1, f_bins=0.0, fdot_bins=1.0, a_rel=0.1, a1_rel=0.2, fddot_hw=150.0 / np.pi)


def piece_estimate(piece: np.ndarray, fs: float):
    """(f, a, k) of one piece of M samples: Hann-windowed FFT peak with log-parabolic refinement (module docstring)."""
    piece = np.asarray(piece, dtype=np.float64)
    M = piece.shape[0]
    m = np.arange(M, dtype=np.float64)
    w = 0.5 - 0.5 * np.cos(2.0 * np.pi * m / M)
    X = np.fft.rfft(piece * w)
    P = X.real**2 + X.imag**2
    k = 1 + int(np.argmax(P[1:M // 2]))                      # bins 1 .. M/2 - 1, lowest k on ties
    lm, l0, lp = np.log(P[k - 1]), np.log(P[k]), np.log(P[k + 1])
    den = lm - 2.0 * l0 + lp
    delta = 0.5 * (lm - lp) / den if den != 0.0 else 0.0
    f = (k + delta) * fs / M
    sinc = np.sin(np.pi * delta) / (np.pi * delta) if delta != 0.0 else 1.0
    lobe = sinc / (1.0 - delta * delta)
    a = 4.0 * np.sqrt(P[k]) / M / lobe
    return f, a, k


def acquire(x: np.ndarray, fs: float, D: int, M: int, spacing: int, **kw):
    """x[B][N] -> dict(est[B][8] = (a_est, f_-1, f_0, f_+1, fdot_est, k_-1, k_0, k_+1), lo[B][D], hi[B][D])."""
    cfg = dict(DEFAULTS)
    cfg.update(kw)
    x = np.asarray(x)
    B, N = x.shape
    if M & (M - 1) or M < 8 or M + 2 * spacing > N or spacing < 1 or D not in (5, 6):
        raise ValueError("invalid acquisition arguments")
    T = N / fs
    est = np.zeros((B, 8))
    lo = np.zeros((B, D))
    hi = np.zeros((B, D))
    for b in range(B):
        fk, ak, kk = [], [], []
        for k in (-1, 0, 1):
            i0 = N // 2 + k * spacing - M // 2
            f, a, kp = piece_estimate(x[b, i0:i0 + M], fs)
            fk.append(f); ak.append(a); kk.append(kp)
        a_est, f_c = ak[1], fk[1]
        fdot = (fk[2] - fk[0]) / (2.0 * spacing / fs)
        est[b] = (a_est, fk[0], fk[1], fk[2], fdot, kk[0], kk[1], kk[2])
        f_hw = max(cfg["f_rel"] * abs(f_c), cfg["f_bins"] * fs / M)
        fdot_hw = cfg["fdot_bins"] * (fs / M) / (spacing / fs)
        lo[b, 0], hi[b, 0] = a_est * (1.0 - cfg["a_rel"]), a_est * (1.0 + cfg["a_rel"])
        lo[b, 1], hi[b, 1] = -cfg["a1_rel"] * a_est / T, cfg["a1_rel"] * a_est / T
        lo[b, 2], hi[b, 2] = -np.pi, np.pi
        lo[b, 3], hi[b, 3] = f_c - f_hw, f_c + f_hw
        lo[b, 4], hi[b, 4] = fdot - fdot_hw, fdot + fdot_hw
        if D == 6:
            lo[b, 5], hi[b, 5] = -cfg["fddot_hw"], cfg["fddot_hw"]
    return {"est": est, "lo": lo, "hi": hi}
