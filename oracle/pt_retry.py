"""fp64 oracle of the run-time range determination and the re-search of doubtful blocks
(PAPER.md:191-199 section 3.1.1 second list, :226-248 section 3.1.3, :252 section 3.1.4).

TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/pt_oracle.c's header).

The paper: the correctness of a block's solution is judged by "the continuity of instantaneous phase and frequency at
the bound of two adjacent data block" (Eq. 8) "within the threshold of noise" (:248); ranges at run time are
extrapolated from a solved block n to block n+1 -- c1 in [phi'^n(T/2), phi'^n(3T/2)], c2 in [phi''^n(T/2)/2,
phi''^n(3T/2)/2] ("the sign will be decided by software automatically"), c4 in c4^n -+ 10 %, c0 a full turn, c3 and c5
keep their ranges (:193-197); when a search fails "the software will automatically adjust parameters range and try to
search again.  The data block will be abandoned after three attempts" (:252).

DESIGN.md reading R25 (the paper gives no thresholds, no enlargement rule, and walks the blocks one by one):
  * all blocks are fitted first (in parallel); then, per attempt a = 1 .. max_attempts:
  * border j (between blocks j and j+1) is BAD if |wrap(phi_{j+1}(-T/2) - phi_j(T/2))| > phi_tol or
    |F_{j+1}(-T/2) - F_j(T/2)| > 2 pi F_tol; a block is DOUBTFUL if every border it has is bad (an isolated wrong block
    spoils both of its borders, its neighbours keep one good border each);
  * a doubtful block b takes new ranges from the nearest block n that is not doubtful (the left one on equal distance;
    k = b - n, the paper's k = 1): with F^n(t) = f + fdot t + fddot t^2/2 and F'^n(t) = fdot + fddot t,
        f    in mid[F^n((k-1/2)T), F^n((k+1/2)T)] -+ g max(half their distance, f_floor)
        fdot in mid[F'^n((k-1/2)T), F'^n((k+1/2)T)] -+ g max(half their distance, fdot_floor)
        a0   in a0^n (1 -+ g a_rel),  phi0 in [-pi, pi],  a1 and fddot keep their ranges,
    g = grow^(a-1) the enlargement of attempt a; the floors keep the paper's interval from collapsing when the
    frequency rate is small; if no block is trusted, the block's own box is widened by `grow` about its centre;
  * the doubtful blocks are fitted again (only they), with the Philox key seed + a * 0x9E3779B97F4A7C15 (mod 2^64) and
    their own block indices; a re-fit always replaces the block's previous solution (:252 "search again");
  * blocks still doubtful after the last attempt get status bit 2 ("abandoned").
"""
from __future__ import annotations

import numpy as np

from . import pt_oracle as _o

GOLDEN = 0x9E3779B97F4A7C15
DEFAULTS = dict(phi_tol=0.5, F_tol=0.5, max_attempts=3, grow=2.0, f_floor=1.0, fdot_floor=1.0, a_rel=0.1)


def doubtful_blocks(per_block: np.ndarray, phi_tol: float, F_tol: float) -> np.ndarray:
    """flags[B] from the border residual columns 8 (phase, rad) and 9 (frequency, rad/s) of the Doppler products."""
    B = per_block.shape[0]
    bad = (np.abs(per_block[:-1, 8]) > phi_tol) | (np.abs(per_block[:-1, 9]) > 2.0 * np.pi * F_tol)   # borders 0..B-2
    flags = np.zeros(B, dtype=bool)
    for b in range(B):
        borders = []
        if b > 0:
            borders.append(bad[b - 1])
        if b < B - 1:
            borders.append(bad[b])
        flags[b] = len(borders) > 0 and all(borders)
    return flags


def extrapolated_box(b: int, flags: np.ndarray, best: np.ndarray, lo_b: np.ndarray, hi_b: np.ndarray, T: float, g: float,
                     grow: float, f_floor: float, fdot_floor: float, a_rel: float):
    """New (lo, hi) of doubtful block b (module docstring)."""
    B, D = best.shape
    lo, hi = lo_b.copy(), hi_b.copy()
    left = [n for n in range(b - 1, -1, -1) if not flags[n]]
    right = [n for n in range(b + 1, B) if not flags[n]]
    if not left and not right:
        c, h = 0.5 * (lo + hi), 0.5 * (hi - lo) * grow
        return c - h, c + h
    if left and (not right or b - left[0] <= right[0] - b):
        n = left[0]
    else:
        n = right[0]
    k = float(b - n)
    a0, f, fdot = best[n, 0], best[n, 3], best[n, 4]
    fddot = best[n, 5] if D == 6 else 0.0
    t1, t2 = (k - 0.5) * T, (k + 0.5) * T
    e1 = f + fdot * t1 + fddot * t1 * t1 / 2.0
    e2 = f + fdot * t2 + fddot * t2 * t2 / 2.0
    d1 = fdot + fddot * t1
    d2 = fdot + fddot * t2
    hw = g * max(abs(e2 - e1) / 2.0, f_floor)
    lo[3], hi[3] = (e1 + e2) / 2.0 - hw, (e1 + e2) / 2.0 + hw
    hw = g * max(abs(d2 - d1) / 2.0, fdot_floor)
    lo[4], hi[4] = (d1 + d2) / 2.0 - hw, (d1 + d2) / 2.0 + hw
    lo[0], hi[0] = a0 * (1.0 - g * a_rel), a0 * (1.0 + g * a_rel)
    if lo[0] > hi[0]:
        lo[0], hi[0] = hi[0], lo[0]
    lo[2], hi[2] = -np.pi, np.pi
    return lo, hi


def refit_doubtful(x, fs, lo, hi, best, best_rss, status, *, NP, generations, F=0.5, CR=0.9, seed=0, strategy=1,
                   objective=0, block_index=None, **kw):
    """Returns dict(best, best_rss, status, lo, hi, attempts[B], flags_per_attempt[list of bool[B]])."""
    cfg = dict(DEFAULTS)
    cfg.update(kw)
    x = np.asarray(x, dtype=np.float32)
    B, N = x.shape
    T = N / fs
    lo, hi = np.array(lo, dtype=np.float64), np.array(hi, dtype=np.float64)
    best = np.array(best, dtype=np.float64)
    best_rss = np.array(best_rss, dtype=np.float64)
    status = np.array(status, dtype=np.uint32)
    bidx = np.arange(B, dtype=np.uint32) if block_index is None else np.asarray(block_index, dtype=np.uint32)
    attempts = np.zeros(B, dtype=np.int32)
    history = []
    flags = np.zeros(B, dtype=bool)
    for a in range(1, int(cfg["max_attempts"]) + 1):
        per_block, _, _ = _o.doppler_products(best, T)
        flags = doubtful_blocks(per_block, cfg["phi_tol"], cfg["F_tol"])
        history.append(flags.copy())
        sel = np.nonzero(flags)[0]
        if sel.size == 0:
            break
        g = cfg["grow"] ** (a - 1)
        new_lo, new_hi = lo.copy(), hi.copy()
        for b in sel:
            new_lo[b], new_hi[b] = extrapolated_box(int(b), flags, best, lo[b], hi[b], T, g, cfg["grow"], cfg["f_floor"],
                                                    cfg["fdot_floor"], cfg["a_rel"])
        lo, hi = new_lo, new_hi
        r = _o.fit_blocks(x[sel], fs, lo[sel], hi[sel], NP=NP, generations=generations, F=F, CR=CR,
                          seed=(seed + a * GOLDEN) % (1 << 64), block_index=bidx[sel], strategy=strategy, objective=objective)
        best[sel], best_rss[sel], status[sel] = r["best"], r["best_rss"], r["status"]
        attempts[sel] += 1
    else:
        per_block, _, _ = _o.doppler_products(best, T)
        flags = doubtful_blocks(per_block, cfg["phi_tol"], cfg["F_tol"])
        history.append(flags.copy())
        status[flags] |= 4
    return {"best": best, "best_rss": best_rss, "status": status, "lo": lo, "hi": hi, "attempts": attempts,
            "flags_per_attempt": history}
