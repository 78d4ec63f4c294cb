"""Thin ctypes binding of ``libpt.so`` (C ABI in ``include/pt.h``): argument marshalling only.

Every function takes torch CUDA tensors (device memory and streams are torch's), passes their data
pointers and the current CUDA stream to the entry point of the same name, and raises ``PtError`` on a
non-zero status.  There is no CPU fallback: if ``libpt.so`` is missing it is built with nvcc; if it cannot
be built or loaded, or no CUDA device is present, the call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import build as _build

_lib = None


class PtError(RuntimeError):
    pass


class DEConfig(C.Structure):
    """Mirror of ``pt_de_config`` (include/pt.h)."""

    _fields_ = [
        ("D", C.c_int32),
        ("NP", C.c_int32),
        ("generations", C.c_int32),
        ("F", C.c_double),
        ("CR", C.c_double),
        ("seed", C.c_uint64),
        ("t0", C.c_double),
        ("strategy", C.c_int32),
        ("objective", C.c_int32),
    ]


class Quant(C.Structure):
    """Mirror of ``pt_quant`` (include/pt.h): s = scale * (code + offset)."""

    _fields_ = [("bits", C.c_int32), ("is_signed", C.c_int32), ("scale", C.c_double), ("offset", C.c_double)]


class AcqConfig(C.Structure):
    """Mirror of ``pt_acq_config`` (include/pt.h)."""

    _fields_ = [("M", C.c_int32), ("spacing", C.c_int32), ("f_rel", C.c_double), ("f_bins", C.c_double),
                ("fdot_bins", C.c_double), ("a_rel", C.c_double), ("a1_rel", C.c_double), ("fddot_hw", C.c_double)]


class RetryConfig(C.Structure):
    """Mirror of ``pt_retry_config`` (include/pt.h)."""

    _fields_ = [("phi_tol", C.c_double), ("F_tol", C.c_double), ("max_attempts", C.c_int32), ("grow", C.c_double),
                ("f_floor", C.c_double), ("fdot_floor", C.c_double), ("a_rel", C.c_double)]


def lib():
    """Load the CUDA library, (re)building it first when the sources changed.  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()        # a no-op when the fingerprint stamp matches; rebuilds a stale library after a source edit
    L = C.CDLL(path)
    p, i32, i64, f64, u64, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_double, C.c_uint64, C.c_size_t
    L.pt_last_error_string.restype = C.c_char_p
    L.pt_version.restype = C.c_char_p
    L.pt_fitness_workspace_bytes.argtypes = [i64, i32, i32, i32]
    L.pt_fitness_workspace_bytes.restype = sz
    L.pt_fitness.argtypes = [p, i64, i32, f64, f64, p, i32, i32, p, p, sz, p]
    L.pt_fitness.restype = i32
    L.pt_objective.argtypes = [p, i64, i32, f64, f64, p, i32, i32, i32, p, p, sz, p]
    L.pt_objective.restype = i32
    L.pt_fit_blocks_workspace_bytes.argtypes = [i64, i32, C.POINTER(DEConfig)]
    L.pt_fit_blocks_workspace_bytes.restype = sz
    L.pt_fit_blocks.argtypes = [p, i64, i32, f64, p, p, p, C.POINTER(DEConfig), p, p, p, p, p, p, sz, p]
    L.pt_fit_blocks.restype = i32
    L.pt_fit_blocks_q.argtypes = [p, C.POINTER(Quant), i64, i64, i32, f64, p, p, p, C.POINTER(DEConfig), p, p, p, p, p, p, sz, p]
    L.pt_fit_blocks_q.restype = i32
    L.pt_unpack_samples.argtypes = [p, C.POINTER(Quant), i64, i64, i32, p, p]
    L.pt_unpack_samples.restype = i32
    L.pt_track_host_q.argtypes = [p, C.POINTER(Quant), i64, i64, i32, f64, p, p, C.POINTER(DEConfig), f64, p, i32, p, p, p, p, p, p]
    L.pt_track_host_q.restype = i32
    L.pt_acquire.argtypes = [p, i64, i32, f64, i32, C.POINTER(AcqConfig), p, p, p, p]
    L.pt_acquire.restype = i32
    L.pt_refit_doubtful_workspace_bytes.argtypes = [i64, i32, C.POINTER(DEConfig)]
    L.pt_refit_doubtful_workspace_bytes.restype = sz
    L.pt_refit_doubtful.argtypes = [p, i64, i32, f64, p, p, p, C.POINTER(DEConfig), C.POINTER(RetryConfig), p, p, p, p, p, sz, p]
    L.pt_refit_doubtful.restype = i32
    L.pt_static_scratch_bytes.argtypes = []
    L.pt_static_scratch_bytes.restype = sz
    L.pt_refit_doubtful_static.argtypes = [p, i64, i32, f64, p, p, p, C.POINTER(DEConfig), C.POINTER(RetryConfig), p, p, p, p, p]
    L.pt_refit_doubtful_static.restype = i32
    L.pt_track_auto_host.argtypes = [p, i64, i32, f64, C.POINTER(DEConfig), C.POINTER(AcqConfig), C.POINTER(RetryConfig), f64, p,
                                     i32, p, p, p, p, p, p, p, p, p]
    L.pt_track_auto_host.restype = i32
    L.pt_fit_blocks_plan.argtypes = [i64, i32, C.POINTER(DEConfig), p]
    L.pt_fit_blocks_plan.restype = i32
    L.pt_fit_blocks_launches.argtypes = [i64, i32, C.POINTER(DEConfig), p, i32]
    L.pt_fit_blocks_launches.restype = i32
    L.pt_doppler_products.argtypes = [p, i64, i32, f64, f64, p, i32, p, p, p, p]
    L.pt_doppler_products.restype = i32
    L.pt_track_host.argtypes = [p, i64, i32, f64, p, p, C.POINTER(DEConfig), f64, p, i32, p, p, p, p, p, p]
    L.pt_track_host.restype = i32
    L.pt_host_cache_release.argtypes = []
    L.pt_host_cache_release.restype = i32
    L.pt_de_draws.argtypes = [p, i64, i32, i32, f64, u64, p, p]
    L.pt_de_draws.restype = i32
    L.pt_init_population.argtypes = [p, p, p, i64, i32, i32, u64, p, p]
    L.pt_init_population.restype = i32
    _lib = L
    return L


def _check(rc: int, what: str):
    if rc != 0:
        raise PtError("%s failed (%d): %s" % (what, rc, lib().pt_last_error_string().decode()))


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dev(t: torch.Tensor, dtype, name: str) -> int:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise PtError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))
    return t.data_ptr()


def default_t0(N: int, fs: float) -> float:
    return -float(N) / (2.0 * float(fs))


STRATEGY_RAND1, STRATEGY_LOCAL_TO_BEST1, STRATEGY_BEST1_JITTER = 1, 2, 3
STRATEGY_RAND1_VEC_DITHER, STRATEGY_RAND1_GEN_DITHER, STRATEGY_EITHER_OR = 4, 5, 6
OBJECTIVE_CHI2, OBJECTIVE_COR = 0, 1


def make_config(*, D: int, NP: int, generations: int, F: float = 0.5, CR: float = 0.9, seed: int = 0,
                t0: float, strategy: int = STRATEGY_RAND1, objective: int = OBJECTIVE_CHI2) -> DEConfig:
    return DEConfig(int(D), int(NP), int(generations), float(F), float(CR), int(seed), float(t0), int(strategy),
                    int(objective))


def pt_fitness(x: torch.Tensor, fs: float, pop: torch.Tensor, t0: float | None = None) -> torch.Tensor:
    """fitness[B][NP] fp32 of pop[B][NP][D] fp32 on x[B][N] fp32 (Eq. 4)."""
    B, N = x.shape
    _, NP, D = pop.shape
    if pop.shape[0] != B:
        raise PtError("pop must be [B][NP][D]")
    if t0 is None:
        t0 = default_t0(N, fs)
    out = torch.empty((B, NP), dtype=torch.float32, device=x.device)
    ws_bytes = lib().pt_fitness_workspace_bytes(B, N, NP, D)
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=x.device) if ws_bytes else None
    rc = lib().pt_fitness(_dev(x, torch.float32, "x"), B, N, float(fs), float(t0), _dev(pop, torch.float32, "pop"), NP, D,
                          out.data_ptr(), ws.data_ptr() if ws is not None else None, ws_bytes, _stream())
    _check(rc, "pt_fitness")
    return out


def pt_objective(x: torch.Tensor, fs: float, pop: torch.Tensor, objective: int, t0: float | None = None) -> torch.Tensor:
    """[B][NP] fp32: Eq. 4 (objective 0) or F_cor - 1/pi of Eq. 5-6 (objective 1) of pop[B][NP][D] on x[B][N]."""
    B, N = x.shape
    _, NP, D = pop.shape
    if pop.shape[0] != B:
        raise PtError("pop must be [B][NP][D]")
    if t0 is None:
        t0 = default_t0(N, fs)
    out = torch.empty((B, NP), dtype=torch.float32, device=x.device)
    ws_bytes = lib().pt_fitness_workspace_bytes(B, N, NP, D)
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=x.device) if ws_bytes else None
    rc = lib().pt_objective(_dev(x, torch.float32, "x"), B, N, float(fs), float(t0), _dev(pop, torch.float32, "pop"), NP, D,
                            int(objective), out.data_ptr(), ws.data_ptr() if ws is not None else None, ws_bytes, _stream())
    _check(rc, "pt_objective")
    return out


def make_quant(bits: int, is_signed: bool, scale: float, offset: float = 0.0) -> Quant:
    return Quant(int(bits), int(bool(is_signed)), float(scale), float(offset))


def pt_unpack_samples(xq: torch.Tensor, N: int, quant: Quant) -> torch.Tensor:
    """xq[B][row_bytes] uint8 (device) -> x[B][N] fp32."""
    B, row_bytes = xq.shape
    x = torch.empty((B, int(N)), dtype=torch.float32, device=xq.device)
    rc = lib().pt_unpack_samples(_dev(xq, torch.uint8, "xq"), C.byref(quant), row_bytes, B, int(N), x.data_ptr(), _stream())
    _check(rc, "pt_unpack_samples")
    return x


def pt_fit_blocks(x: torch.Tensor, fs: float, lo: torch.Tensor, hi: torch.Tensor, cfg: DEConfig, *,
                  block_index: torch.Tensor | None = None, want_pop: bool = False, quant: Quant | None = None,
                  N: int | None = None) -> dict:
    """DE fit of every block; returns dict(best[B][D] f64, best_rss[B] f32, status[B] i32-view of u32
    [, final_pop[B][NP][D] f32, final_fit[B][NP] f32]).  With ``quant`` x is uint8 [B][row_bytes] of packed samples
    (pt_fit_blocks_q) and ``N`` is the number of samples per block."""
    if quant is None:
        B, N = x.shape
    else:
        B, row_bytes = x.shape
        N = int(N)
    D, NP = cfg.D, cfg.NP
    if tuple(lo.shape) != (B, D) or tuple(hi.shape) != (B, D):
        raise PtError("lo and hi must be [B][D]")
    dev = x.device
    best = torch.empty((B, D), dtype=torch.float64, device=dev)
    best_rss = torch.empty(B, dtype=torch.float32, device=dev)
    status = torch.empty(B, dtype=torch.int32, device=dev)
    fpop = torch.empty((B, NP, D), dtype=torch.float32, device=dev) if want_pop else None
    ffit = torch.empty((B, NP), dtype=torch.float32, device=dev) if want_pop else None
    ws_bytes = lib().pt_fit_blocks_workspace_bytes(B, N, C.byref(cfg))
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev) if ws_bytes else None
    bidx = None if block_index is None else _dev(block_index, torch.int32, "block_index")
    tail = (_dev(lo, torch.float64, "lo"), _dev(hi, torch.float64, "hi"), bidx, C.byref(cfg), best.data_ptr(),
            best_rss.data_ptr(), status.data_ptr(), fpop.data_ptr() if want_pop else None,
            ffit.data_ptr() if want_pop else None, ws.data_ptr() if ws is not None else None, ws_bytes, _stream())
    if quant is None:
        rc = lib().pt_fit_blocks(_dev(x, torch.float32, "x"), B, N, float(fs), *tail)
    else:
        rc = lib().pt_fit_blocks_q(_dev(x, torch.uint8, "xq"), C.byref(quant), row_bytes, B, N, float(fs), *tail)
    _check(rc, "pt_fit_blocks")
    out = {"best": best, "best_rss": best_rss, "status": status}
    if want_pop:
        out["final_pop"] = fpop
        out["final_fit"] = ffit
    return out


def make_acq_config(*, M: int, spacing: int, f_rel: float = 0.1, f_bins: float = 0.0, fdot_bins: float = 1.0,
                    a_rel: float = 0.1, a1_rel: float = 0.2, fddot_hw: float = 47.746482927568600) -> AcqConfig:
    """Defaults are the paper's percentages; fddot_hw = 150/pi is c3 in [-50, 50]."""
    return AcqConfig(int(M), int(spacing), float(f_rel), float(f_bins), float(fdot_bins), float(a_rel), float(a1_rel),
                     float(fddot_hw))


def pt_acquire(x: torch.Tensor, fs: float, D: int, acq: AcqConfig) -> dict:
    """Initial ranges of every block: dict(est[B][8], lo[B][D], hi[B][D]) fp64 on the device."""
    B, N = x.shape
    dev = x.device
    est = torch.empty((B, 8), dtype=torch.float64, device=dev)
    lo = torch.empty((B, int(D)), dtype=torch.float64, device=dev)
    hi = torch.empty((B, int(D)), dtype=torch.float64, device=dev)
    rc = lib().pt_acquire(_dev(x, torch.float32, "x"), B, N, float(fs), int(D), C.byref(acq), est.data_ptr(), lo.data_ptr(),
                          hi.data_ptr(), _stream())
    _check(rc, "pt_acquire")
    return {"est": est, "lo": lo, "hi": hi}


def make_retry_config(*, phi_tol: float, F_tol: float, max_attempts: int = 3, grow: float = 2.0, f_floor: float = 1.0,
                      fdot_floor: float = 1.0, a_rel: float = 0.1) -> RetryConfig:
    return RetryConfig(float(phi_tol), float(F_tol), int(max_attempts), float(grow), float(f_floor), float(fdot_floor),
                       float(a_rel))


def pt_refit_doubtful(x: torch.Tensor, fs: float, lo: torch.Tensor, hi: torch.Tensor, cfg: DEConfig, retry: RetryConfig,
                      fit: dict, *, block_index: torch.Tensor | None = None) -> torch.Tensor:
    """Continuity check + re-search of doubtful blocks; updates lo, hi and fit["best"/"best_rss"/"status"] in place and
    returns attempts[B] int32."""
    B, N = x.shape
    attempts = torch.empty(B, dtype=torch.int32, device=x.device)
    ws_bytes = lib().pt_refit_doubtful_workspace_bytes(B, N, C.byref(cfg))
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=x.device)
    bidx = None if block_index is None else _dev(block_index, torch.int32, "block_index")
    rc = lib().pt_refit_doubtful(_dev(x, torch.float32, "x"), B, N, float(fs), _dev(lo, torch.float64, "lo"),
                                 _dev(hi, torch.float64, "hi"), bidx, C.byref(cfg), C.byref(retry),
                                 _dev(fit["best"], torch.float64, "best"), _dev(fit["best_rss"], torch.float32, "best_rss"),
                                 _dev(fit["status"], torch.int32, "status"), attempts.data_ptr(), ws.data_ptr(), ws_bytes,
                                 _stream())
    _check(rc, "pt_refit_doubtful")
    return attempts


def pt_refit_doubtful_static(x: torch.Tensor, fs: float, lo: torch.Tensor, hi: torch.Tensor, cfg: DEConfig, retry: RetryConfig,
                             fit: dict, attempts: torch.Tensor, *, block_index: torch.Tensor | None = None) -> torch.Tensor:
    """pt_refit_doubtful without a workspace: the scratch is the library's static device array (include/pt.h), nothing is
    allocated -- here neither: `attempts` [B] int32 is the caller's.  Returns `attempts`."""
    B, N = x.shape
    bidx = None if block_index is None else _dev(block_index, torch.int32, "block_index")
    rc = lib().pt_refit_doubtful_static(_dev(x, torch.float32, "x"), B, N, float(fs), _dev(lo, torch.float64, "lo"),
                                        _dev(hi, torch.float64, "hi"), bidx, C.byref(cfg), C.byref(retry),
                                        _dev(fit["best"], torch.float64, "best"), _dev(fit["best_rss"], torch.float32, "best_rss"),
                                        _dev(fit["status"], torch.int32, "status"), _dev(attempts, torch.int32, "attempts"),
                                        _stream())
    _check(rc, "pt_refit_doubtful_static")
    return attempts


def pt_fit_blocks_plan(B: int, N: int, cfg: DEConfig) -> dict:
    out = (C.c_int32 * 8)()
    _check(lib().pt_fit_blocks_plan(B, N, C.byref(cfg), out), "pt_fit_blocks_plan")
    return dict(grid=out[0], threads=out[1], smem=out[2], resident=out[3], cands_per_thread=out[4], ctas_per_sm=out[5],
                cluster=out[6], tail_cluster=out[7])


def pt_fit_blocks_launches(B: int, N: int, cfg: DEConfig) -> list:
    """The DE-kernel launches of pt_fit_blocks: [dict(first, blocks, grid, threads, cluster), ...] (include/pt.h)."""
    out = (C.c_int32 * (5 * 16))()
    n = lib().pt_fit_blocks_launches(B, N, C.byref(cfg), out, 16)
    _check(min(n, 0), "pt_fit_blocks_launches")
    return [dict(first=out[5 * k], blocks=out[5 * k + 1], grid=out[5 * k + 2], threads=out[5 * k + 3], cluster=out[5 * k + 4])
            for k in range(min(n, 16))]


def pt_doppler_products(best: torch.Tensor, T: float, los_scale: float = 0.0, blocks_per_interval=()):
    """(per_block[B][10], total_phase[B], [interval tensors [floor(B/m)][2]]), all fp64 on the device."""
    B, D = best.shape
    dev = best.device
    m = [int(v) for v in blocks_per_interval]
    per_block = torch.empty((B, 10), dtype=torch.float64, device=dev)
    total = torch.empty(B, dtype=torch.float64, device=dev)
    outs = [torch.empty((B // v, 2), dtype=torch.float64, device=dev) for v in m]
    m_arr = (C.c_int32 * max(len(m), 1))(*m)
    ptrs = (C.c_void_p * max(len(m), 1))(*[o.data_ptr() if o.numel() else None for o in outs])
    rc = lib().pt_doppler_products(_dev(best, torch.float64, "best"), B, D, float(T), float(los_scale), m_arr, len(m),
                                   per_block.data_ptr(), total.data_ptr(), ptrs, _stream())
    _check(rc, "pt_doppler_products")
    return per_block, total, outs


def pt_track_host(x, fs: float, lo, hi, cfg: DEConfig, los_scale: float = 0.0, blocks_per_interval=(),
                  quant: Quant | None = None, N: int | None = None):
    """Whole hot path on HOST tensors (CPU torch tensors, ideally pinned): H2D, fit, products, D2H.  With ``quant``
    x is uint8 [B][row_bytes] of packed samples (pt_track_host_q) and ``N`` the samples per block."""
    if quant is None:
        B, N = x.shape
    else:
        B, row_bytes = x.shape
        N = int(N)
    D = cfg.D
    for t, dt, nm in ((x, torch.float32 if quant is None else torch.uint8, "x"), (lo, torch.float64, "lo"), (hi, torch.float64, "hi")):
        if t.is_cuda or t.dtype != dt or not t.is_contiguous():
            raise PtError("%s must be a contiguous host tensor of dtype %s" % (nm, dt))
    m = [int(v) for v in blocks_per_interval]
    best = torch.empty((B, D), dtype=torch.float64)
    best_rss = torch.empty(B, dtype=torch.float32)
    status = torch.empty(B, dtype=torch.int32)
    per_block = torch.empty((B, 10), dtype=torch.float64)
    total = torch.empty(B, dtype=torch.float64)
    outs = [torch.empty((B // v, 2), dtype=torch.float64) for v in m]
    m_arr = (C.c_int32 * max(len(m), 1))(*m)
    ptrs = (C.c_void_p * max(len(m), 1))(*[o.data_ptr() if o.numel() else None for o in outs])
    tail = (B, N, float(fs), lo.data_ptr(), hi.data_ptr(), C.byref(cfg), float(los_scale), m_arr, len(m), best.data_ptr(),
            best_rss.data_ptr(), status.data_ptr(), per_block.data_ptr(), total.data_ptr(), ptrs)
    if quant is None:
        rc = lib().pt_track_host(x.data_ptr(), *tail)
    else:
        rc = lib().pt_track_host_q(x.data_ptr(), C.byref(quant), row_bytes, *tail)
    _check(rc, "pt_track_host")
    return {"best": best, "best_rss": best_rss, "status": status, "per_block": per_block, "total_phase": total,
            "intervals": outs}


def pt_host_cache_release() -> None:
    """Free the per-device memory pools and streams the *_host entry points keep between calls."""
    _check(lib().pt_host_cache_release(), "pt_host_cache_release")


def pt_track_auto_host(x, fs: float, cfg: DEConfig, acq: AcqConfig, retry: RetryConfig | None = None,
                       los_scale: float = 0.0, blocks_per_interval=()):
    """The whole process flow on HOST tensors with no caller ranges: H2D, acquisition, fit, re-search (if ``retry``),
    products, D2H."""
    B, N = x.shape
    D = cfg.D
    if x.is_cuda or x.dtype != torch.float32 or not x.is_contiguous():
        raise PtError("x must be a contiguous host tensor of dtype float32")
    m = [int(v) for v in blocks_per_interval]
    lo = torch.empty((B, D), dtype=torch.float64)
    hi = torch.empty((B, D), dtype=torch.float64)
    best = torch.empty((B, D), dtype=torch.float64)
    best_rss = torch.empty(B, dtype=torch.float32)
    status = torch.empty(B, dtype=torch.int32)
    attempts = torch.zeros(B, dtype=torch.int32)
    per_block = torch.empty((B, 10), dtype=torch.float64)
    total = torch.empty(B, dtype=torch.float64)
    outs = [torch.empty((B // v, 2), dtype=torch.float64) for v in m]
    m_arr = (C.c_int32 * max(len(m), 1))(*m)
    ptrs = (C.c_void_p * max(len(m), 1))(*[o.data_ptr() if o.numel() else None for o in outs])
    rc = lib().pt_track_auto_host(x.data_ptr(), B, N, float(fs), C.byref(cfg), C.byref(acq),
                                  C.byref(retry) if retry is not None else None, float(los_scale), m_arr, len(m),
                                  lo.data_ptr(), hi.data_ptr(), best.data_ptr(), best_rss.data_ptr(), status.data_ptr(),
                                  attempts.data_ptr(), per_block.data_ptr(), total.data_ptr(), ptrs)
    _check(rc, "pt_track_auto_host")
    return {"lo": lo, "hi": hi, "best": best, "best_rss": best_rss, "status": status, "attempts": attempts,
            "per_block": per_block, "total_phase": total, "intervals": outs}


def pt_de_draws(query: torch.Tensor, NP: int, D: int, CR: float, seed: int) -> torch.Tensor:
    """query[Q][3] int32 (block_index, generation, candidate) -> [Q][5] int32 (r1, r2, r3, jrand, mask)."""
    Q = query.shape[0]
    out = torch.empty((Q, 5), dtype=torch.int32, device=query.device)
    rc = lib().pt_de_draws(_dev(query, torch.int32, "query"), Q, NP, D, float(CR), int(seed), out.data_ptr(), _stream())
    _check(rc, "pt_de_draws")
    return out


def pt_init_population(lo: torch.Tensor, hi: torch.Tensor, NP: int, seed: int,
                       block_index: torch.Tensor | None = None) -> torch.Tensor:
    B, D = lo.shape
    out = torch.empty((B, NP, D), dtype=torch.float64, device=lo.device)
    bidx = None if block_index is None else _dev(block_index, torch.int32, "block_index")
    rc = lib().pt_init_population(_dev(lo, torch.float64, "lo"), _dev(hi, torch.float64, "hi"), bidx, B, NP, D, int(seed),
                                  out.data_ptr(), _stream())
    _check(rc, "pt_init_population")
    return out
