"""ctypes marshalling for ``oracle/pt_oracle.c`` (test infrastructure; see that file's header).

No arithmetic of the method lives here: every function below copies numpy arrays in and out of
the C oracle.  ``build()`` compiles the C file with gcc (``-ffp-contract=off`` so that no
multiply-add is fused and every fp64 operation rounds as written).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pt_oracle.c")
_LIB = os.path.join(_HERE, "libpt_oracle.so")
_lock = threading.Lock()
_lib = None


class _DEConfig(C.Structure):
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


def build(force: bool = False) -> str:
    """Compile the C oracle into ``oracle/libpt_oracle.so`` (no-op when up to date)."""
    with _lock:
        if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
            return _LIB
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
        return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = C.CDLL(_LIB)
    p = C.c_void_p
    lib.pto_num_threads.restype = C.c_int
    lib.pto_philox4x32_10.argtypes = [p, p, p]
    lib.pto_cr32.argtypes = [C.c_double]
    lib.pto_cr32.restype = C.c_uint32
    lib.pto_de_draws.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_int32, C.c_int32, C.c_uint32, p]
    lib.pto_indices_from_words.argtypes = [p, C.c_uint32, C.c_int32, C.c_int32, p]
    lib.pto_init_uniforms.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_int32, p]
    lib.pto_model.argtypes = [p, C.c_int32, C.c_double]
    lib.pto_model.restype = C.c_double
    lib.pto_rss.argtypes = [p, C.c_int32, C.c_double, C.c_double, p, C.c_int32]
    lib.pto_rss.restype = C.c_double
    lib.pto_fitness.argtypes = [p, C.c_int64, C.c_int32, C.c_double, C.c_double, p, C.c_int32, C.c_int32, p]
    lib.pto_fitness_obj.argtypes = [p, C.c_int64, C.c_int32, C.c_double, C.c_double, p, C.c_int32, C.c_int32, C.c_int32, p]
    lib.pto_cor.argtypes = [p, C.c_int32, C.c_double, C.c_double, p, C.c_int32]
    lib.pto_cor.restype = C.c_double
    lib.pto_fcor_of_cor.argtypes = [C.c_double]
    lib.pto_fcor_of_cor.restype = C.c_double
    lib.pto_aux_uniforms.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, p]
    lib.pto_de_trial.argtypes = [C.POINTER(_DEConfig), C.c_uint32, C.c_uint32, C.c_uint32, p, C.c_int32, p, p, p]
    lib.pto_fit_blocks.argtypes = [p, C.c_int64, C.c_int32, C.c_double, p, p, C.POINTER(_DEConfig), p, p, p, p, p, p, p]
    lib.pto_fit_blocks.restype = C.c_int32
    lib.pto_unpack_samples.argtypes = [p, C.c_int64, C.c_int64, C.c_int32, C.c_int32, C.c_int32, C.c_double, C.c_double, p]
    lib.pto_unpack_samples.restype = C.c_int32
    lib.pto_doppler_products.argtypes = [p, C.c_int64, C.c_int32, C.c_double, C.c_double, p, C.c_int32, p, p, p]
    lib.pto_doppler_products.restype = C.c_int32
    _lib = lib
    return lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(_load().pto_num_threads())


def default_t0(N: int, fs: float) -> float:
    return -float(N) / (2.0 * float(fs))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    _load().pto_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def cr32(CR: float) -> int:
    return int(_load().pto_cr32(float(CR)))


def de_draws(seed: int, b: int, g: int, i: int, NP: int, D: int, CR: float):
    """(r1, r2, r3, jrand, mask) of candidate i, generation g >= 1, block b."""
    out = np.zeros(5, dtype=np.int32)
    lib = _load()
    lib.pto_de_draws(int(seed), int(b), int(g), int(i), int(NP), int(D), lib.pto_cr32(float(CR)), _ptr(out))
    return tuple(int(v) for v in out)


def indices_from_words(words, i: int, NP: int, D: int):
    """(r1, r2, r3, jrand) from the four raw 32-bit words of slot 0."""
    w = np.asarray(words, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.int32)
    _load().pto_indices_from_words(_ptr(w), int(i), int(NP), int(D), _ptr(out))
    return tuple(int(v) for v in out)


def init_uniforms(seed: int, b: int, i: int, D: int):
    u = np.zeros(8, dtype=np.float64)
    _load().pto_init_uniforms(int(seed), int(b), int(i), int(D), _ptr(u))
    return u[:D].copy()


def model(theta, t: float) -> float:
    th = np.ascontiguousarray(theta, dtype=np.float64)
    return float(_load().pto_model(_ptr(th), int(th.shape[0]), float(t)))


def rss(x, fs: float, theta, t0: float | None = None) -> float:
    x = np.ascontiguousarray(x, dtype=np.float32)
    th = np.ascontiguousarray(theta, dtype=np.float64)
    N = int(x.shape[0])
    if t0 is None:
        t0 = default_t0(N, fs)
    return float(_load().pto_rss(_ptr(x), N, float(fs), float(t0), _ptr(th), int(th.shape[0])))


def cor(x, fs: float, theta, t0: float | None = None) -> float:
    """Correlation sum of Eq. 5-6 (constant amplitude theta[0])."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    th = np.ascontiguousarray(theta, dtype=np.float64)
    N = int(x.shape[0])
    if t0 is None:
        t0 = default_t0(N, fs)
    return float(_load().pto_cor(_ptr(x), N, float(fs), float(t0), _ptr(th), int(th.shape[0])))


def fcor_of_cor(c: float) -> float:
    """Eq. 5: 1 / (arctan(cor) + pi/2)."""
    return float(_load().pto_fcor_of_cor(float(c)))


def aux_uniforms(seed: int, b: int, g: int, i: int):
    """(jitter[8], per-vector, per-generation) uniforms of the strategies 3-6."""
    u = np.zeros(10, dtype=np.float64)
    _load().pto_aux_uniforms(int(seed), int(b), int(g), int(i), _ptr(u))
    return u[:8].copy(), float(u[8]), float(u[9])


def de_trial(pop, ibest: int, lo, hi, *, b: int, g: int, i: int, F: float, CR: float, seed: int, strategy: int):
    """Trial vector of candidate i in generation g built from the population pop[NP][D]."""
    pop = np.ascontiguousarray(pop, dtype=np.float64)
    lo = np.ascontiguousarray(lo, dtype=np.float64)
    hi = np.ascontiguousarray(hi, dtype=np.float64)
    NP, D = pop.shape
    cfg = _DEConfig(D, NP, 0, float(F), float(CR), int(seed), 0.0, int(strategy), 0)
    out = np.zeros(D, dtype=np.float64)
    _load().pto_de_trial(C.byref(cfg), int(b), int(g), int(i), _ptr(pop), int(ibest), _ptr(lo), _ptr(hi), _ptr(out))
    return out


def fitness(x, fs: float, pop, t0: float | None = None, objective: int = 0):
    """x[B][N] fp32, pop[B][NP][D] fp32 -> objective[B][NP] fp64 (0: Eq. 4 chi^2, 1: Eq. 5 F_cor)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    pop = np.ascontiguousarray(pop, dtype=np.float32)
    B, N = x.shape
    _, NP, D = pop.shape
    assert pop.shape[0] == B
    if t0 is None:
        t0 = default_t0(N, fs)
    out = np.zeros((B, NP), dtype=np.float64)
    _load().pto_fitness_obj(_ptr(x), B, N, float(fs), float(t0), _ptr(pop), NP, D, int(objective), _ptr(out))
    return out


def fit_blocks(x, fs: float, lo, hi, *, NP: int, generations: int, F: float = 0.5, CR: float = 0.9, seed: int = 0,
               t0: float | None = None, block_index=None, want_pop: bool = False, want_trace: bool = False,
               strategy: int = 1, objective: int = 0):
    """DE fit of every block.  Returns a dict: best[B][D], best_rss[B], status[B] and, on request,
    final_pop[B][NP][D], final_fit[B][NP], trace[B][G+1]."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    lo = np.ascontiguousarray(lo, dtype=np.float64)
    hi = np.ascontiguousarray(hi, dtype=np.float64)
    B, N = x.shape
    D = int(lo.shape[1])
    assert lo.shape == (B, D) and hi.shape == (B, D)
    if t0 is None:
        t0 = default_t0(N, fs)
    cfg = _DEConfig(D, int(NP), int(generations), float(F), float(CR), int(seed), float(t0), int(strategy), int(objective))
    best = np.zeros((B, D), dtype=np.float64)
    best_rss = np.zeros(B, dtype=np.float64)
    status = np.zeros(B, dtype=np.uint32)
    fpop = np.zeros((B, NP, D), dtype=np.float64) if want_pop else None
    ffit = np.zeros((B, NP), dtype=np.float64) if want_pop else None
    trace = np.zeros((B, generations + 1), dtype=np.float64) if want_trace else None
    bidx = None if block_index is None else np.ascontiguousarray(block_index, dtype=np.uint32)
    rc = _load().pto_fit_blocks(_ptr(x), B, N, float(fs), _ptr(lo), _ptr(hi), C.byref(cfg), _ptr(bidx), _ptr(best),
                                _ptr(best_rss), _ptr(status), _ptr(fpop), _ptr(ffit), _ptr(trace))
    if rc != 0:
        raise ValueError("pto_fit_blocks: invalid argument")
    out = {"best": best, "best_rss": best_rss, "status": status}
    if want_pop:
        out["final_pop"] = fpop
        out["final_fit"] = ffit
    if want_trace:
        out["trace"] = trace
    return out


def unpack_samples(xq, N: int, bits: int, is_signed: bool, scale: float, offset: float):
    """xq[B][row_bytes] uint8 -> x[B][N] fp32, s = scale (code + offset) (Table 3 sample formats; reading R23)."""
    xq = np.ascontiguousarray(xq, dtype=np.uint8)
    B, row_bytes = xq.shape
    x = np.zeros((B, int(N)), dtype=np.float32)
    rc = _load().pto_unpack_samples(_ptr(xq), row_bytes, B, int(N), int(bits), int(bool(is_signed)), float(scale),
                                    float(offset), _ptr(x))
    if rc != 0:
        raise ValueError("pto_unpack_samples: invalid argument")
    return x


def doppler_products(best, T: float, los_scale: float = 0.0, blocks_per_interval=()):
    """Returns (per_block[B][10], total_phase[B], [interval arrays [floor(B/m)][2]])."""
    best = np.ascontiguousarray(best, dtype=np.float64)
    B, D = best.shape
    m = np.ascontiguousarray(blocks_per_interval, dtype=np.int32)
    per_block = np.zeros((B, 10), dtype=np.float64)
    total = np.zeros(B, dtype=np.float64)
    outs = [np.zeros((max(B // int(v), 0), 2), dtype=np.float64) for v in m]
    ptrs = (C.c_void_p * max(len(outs), 1))(*[o.ctypes.data for o in outs])
    rc = _load().pto_doppler_products(_ptr(best), B, D, float(T), float(los_scale), _ptr(m), len(outs),
                                      _ptr(per_block), _ptr(total), C.cast(ptrs, C.c_void_p))
    if rc != 0:
        raise ValueError("pto_doppler_products: invalid argument")
    return per_block, total, outs
