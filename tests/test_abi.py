"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol include/pt.h declares.
No compute call is made here (there is no GPU on the CPU test box); argument validation that happens before
any CUDA call is checked through the real entry points."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1906_10598_b200 import build
    return build.build()


def _declared_symbols():
    with open(os.path.join(ROOT, "include", "pt.h")) as fh:
        text = fh.read()
    names = re.findall(r"PT_API\s+[\w\s\*]+?\b(pt_\w+)\s*\(", text)
    assert len(names) >= 10
    return sorted(set(names))


def test_header_declares_the_north_star_entry_points():
    names = _declared_symbols()
    for must in ("pt_fitness", "pt_fit_blocks", "pt_doppler_products", "pt_last_error_string"):
        assert must in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = C.CDLL(lib_path)
    for name in _declared_symbols():
        assert hasattr(lib, name), name


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "pt.h"\nint main(void){ pt_de_config c; c.D = 5; return (int)sizeof(c) - (int)sizeof(c); }\n')
    import subprocess
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src), "-o",
                    str(tmp_path / "t.o")], check=True)


def test_struct_layouts_match_the_binding(tmp_path):
    """sizeof / offsetof of pt_de_config and pt_quant as gcc lays them out from include/pt.h = the ctypes mirrors."""
    import subprocess
    from paper_1906_10598_b200.pt import AcqConfig, DEConfig, Quant, RetryConfig
    classes = (DEConfig, Quant, AcqConfig, RetryConfig)
    fields = {"pt_de_config": [f for f, _ in DEConfig._fields_], "pt_quant": [f for f, _ in Quant._fields_],
              "pt_acq_config": [f for f, _ in AcqConfig._fields_], "pt_retry_config": [f for f, _ in RetryConfig._fields_]}
    body = ['#include <stdio.h>', '#include <stddef.h>', '#include "pt.h"', 'int main(void){']
    for st, names in fields.items():
        body.append('printf("%%zu", sizeof(%s));' % st)
        for f in names:
            body.append('printf(" %%zu", offsetof(%s, %s));' % (st, f))
        body.append('printf("\\n");')
    body.append('return 0;}')
    src = tmp_path / "layout.c"
    src.write_text("\n".join(body))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    lines = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.strip().splitlines()
    for line, (st, names), cls in zip(lines, fields.items(), classes):
        nums = [int(v) for v in line.split()]
        assert nums[0] == C.sizeof(cls), st
        assert nums[1:] == [getattr(cls, f).offset for f in names], st
    assert C.sizeof(DEConfig) == 56 and DEConfig.strategy.offset == 48 and DEConfig.objective.offset == 52


def test_argument_validation_needs_no_gpu(lib_path):
    from paper_1906_10598_b200 import pt
    L = pt.lib()
    cfg = pt.make_config(D=5, NP=60, generations=10, t0=-0.5)
    dummy = C.c_void_p(256)
    # null pointers
    assert L.pt_fit_blocks(None, 1, 1000, 1000.0, dummy, dummy, None, C.byref(cfg), dummy, dummy, dummy, None, None,
                           None, 0, None) == -1
    assert b"null" in L.pt_last_error_string()
    # N odd / too small, D, NP, F, CR
    def call(N=1000, cfg=cfg, fs=1000.0):
        return L.pt_fit_blocks(dummy, 1, N, fs, dummy, dummy, None, C.byref(cfg), dummy, dummy, dummy, None, None, None,
                               0, None)
    assert call(N=1001) == -1
    assert call(N=6) == -1
    assert call(fs=0.0) == -1
    assert call(cfg=pt.make_config(D=4, NP=60, generations=1, t0=0.0)) == -1
    assert call(cfg=pt.make_config(D=5, NP=3, generations=1, t0=0.0)) == -1
    assert call(cfg=pt.make_config(D=5, NP=60, generations=-1, t0=0.0)) == -1
    assert call(cfg=pt.make_config(D=5, NP=60, generations=1, F=2.5, t0=0.0)) == -1
    assert call(cfg=pt.make_config(D=5, NP=60, generations=1, CR=1.5, t0=0.0)) == -1
    assert call(cfg=pt.make_config(D=5, NP=4096, generations=1, t0=0.0)) == -2       # beyond PT_MAX_NP
    assert call(N=(1 << 24) + 2) == -2                                                # beyond PT_MAX_N
    assert L.pt_fitness(dummy, 1, 1000, 1000.0, -0.5, dummy, 60, 7, dummy, None, 0, None) == -1
    assert L.pt_doppler_products(dummy, 0, 5, 1.0, 0.0, None, 0, dummy, dummy, None, None) == -1
    assert L.pt_doppler_products(dummy, 4, 5, -1.0, 0.0, None, 0, dummy, dummy, None, None) == -1
    assert L.pt_version().startswith(b"pt ")
    # widened rows: objective / strategy / quantised input are validated before any CUDA call
    assert L.pt_objective(dummy, 1, 1000, 1000.0, -0.5, dummy, 60, 5, 2, dummy, None, 0, None) == -1
    assert call(cfg=pt.make_config(D=5, NP=60, generations=1, t0=0.0, strategy=7)) == -1
    assert call(cfg=pt.make_config(D=5, NP=60, generations=1, t0=0.0, objective=3)) == -1
    q = pt.make_quant(8, True, 1.0)
    assert L.pt_fit_blocks_q(None, C.byref(q), 1000, 1, 1000, 1000.0, dummy, dummy, None, C.byref(cfg), dummy, dummy, dummy,
                             None, None, None, 0, None) == -1
    assert L.pt_fit_blocks_q(dummy, C.byref(pt.make_quant(3, True, 1.0)), 1000, 1, 1000, 1000.0, dummy, dummy, None,
                             C.byref(cfg), dummy, dummy, dummy, None, None, None, 0, None) == -1
    assert L.pt_fit_blocks_q(dummy, C.byref(q), 999, 1, 1000, 1000.0, dummy, dummy, None, C.byref(cfg), dummy, dummy, dummy,
                             None, None, None, 0, None) == -1            # row shorter than N samples
    assert L.pt_unpack_samples(dummy, C.byref(q), 10, 1, 0, dummy, None) == -1


def test_plan_is_computable_without_gpu(lib_path):
    from paper_1906_10598_b200 import pt
    cfg = pt.make_config(D=5, NP=128, generations=1000, t0=-0.5)
    plan = pt.pt_fit_blocks_plan(3600, 16000, cfg)
    assert plan["resident"] == 1 and plan["grid"] >= 148 and plan["threads"] % 32 == 0
    assert plan["smem"] <= 232448


@pytest.mark.parametrize("B,N,NP,D", [(3600, 16000, 128, 5), (36000, 10000, 128, 6), (1024, 1024, 32, 5), (1024, 1024, 128, 5),
                                      (1024, 4096, 512, 5), (1024, 16384, 128, 5), (1024, 65536, 256, 5), (148, 400000, 400, 6),
                                      (60, 10000, 100, 5), (1, 1000, 60, 5), (149, 16000, 128, 5), (296, 16000, 128, 5),
                                      (297, 16000, 128, 5), (443, 10000, 128, 6), (593, 4096, 64, 5), (7, 8, 4, 5)])
def test_launch_list_covers_every_block_once_with_full_grids(lib_path, B, N, NP, D):
    """Host logic of pt_fit_blocks (run_launch_list in csrc/pt_api.cu; no device needed: the plan of a B200).  The launches are
    contiguous, cover blocks 0..B-1 exactly once, never over-subscribe the SMs, and every launch but the last has an exactly full
    grid -- except blocks so short that a generation is bound by the DE step (NP N <= 2^19), whose remainder stays one round;
    blocks with NP N <= 2^18 run on CTAs of 128 threads, eight per SM."""
    from paper_1906_10598_b200 import pt
    cfg = pt.make_config(D=D, NP=NP, generations=10, t0=-0.5 * N / 1000.0)
    plan = pt.pt_fit_blocks_plan(B, N, cfg)
    launches = pt.pt_fit_blocks_launches(B, N, cfg)
    assert 1 <= len(launches) <= 6
    nxt = 0
    for k, ln in enumerate(launches):
        assert ln["first"] == nxt and ln["blocks"] >= 1
        nxt += ln["blocks"]
        assert ln["threads"] in (128, 256, 512, 1024) and 1 <= ln["cluster"] <= 8
        cps = 1024 // ln["threads"]
        assert ln["grid"] <= 148 * cps and ln["grid"] % ln["cluster"] == 0
        if ln["cluster"] > 1:
            assert ln["grid"] == min(ln["blocks"], 148 // ln["cluster"]) * ln["cluster"] or ln["grid"] == ln["blocks"] * ln["cluster"]
        elif plan["resident"] and k + 1 < len(launches):
            assert ln["grid"] == 148 * cps and ln["blocks"] % ln["grid"] == 0           # whole rounds of an exactly full grid
    assert nxt == B
    assert launches[0]["threads"] == plan["threads"] and launches[0]["grid"] == plan["grid"]
    if NP * N <= (1 << 18) and B > 148 * 4:
        assert launches[0]["threads"] == 128
    if B >= 148 * 4 and NP * N > (1 << 19) and plan["resident"]:
        tail = sum(ln["blocks"] for ln in launches[1:])
        assert tail < 148 * (1024 // launches[0]["threads"])                                  # the first launch takes all whole rounds


def test_slices_fill_the_threads_in_whole_rounds(lib_path):
    """choose_slices: NP x S work items over the CTA's threads.  Seen from outside through the shared-memory size of the plan
    (part[S][NP] fp64): NP = 400 on 1024 threads takes S = 5 (2000 items, two rounds) on the streamed paper-shaped blocks."""
    from paper_1906_10598_b200 import pt
    cfg = pt.make_config(D=6, NP=400, generations=10, t0=-1.0)
    plan = pt.pt_fit_blocks_plan(148, 400000, cfg)
    assert plan["resident"] == 0 and plan["threads"] == 1024
    fixed = 128 + 3 * 8192 * 4 + 2 * 400 * 6 * 8 + 3 * 8 * 8 + 400 * 8          # barriers, ring, populations, box, fit
    assert plan["smem"] - fixed == 400 * 5 * 8


def test_product_path_has_no_oracle_import():
    """The package must not import, read or run anything under oracle/ (the oracle is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_1906_10598_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, f)) as fh:
                    text = fh.read()
                assert "import oracle" not in text and "from oracle" not in text and "pt_oracle" not in text, f


def test_lib_rebuilds_a_stale_library(monkeypatch):
    """pt.lib() goes through build.build() every time (a no-op when the fingerprint stamp matches), so a source edit can never
    leave tests running an old binary."""
    from paper_1906_10598_b200 import build, pt
    calls = []
    real = build.build

    def spy(*a, **k):
        calls.append(1)
        return real(*a, **k)

    monkeypatch.setattr(build, "build", spy)
    monkeypatch.setattr(pt, "_lib", None)
    pt.lib()
    assert calls, "pt.lib() must call build.build()"
    # the stamp makes the second build a no-op: the library file is not rewritten
    before = os.path.getmtime(build.LIB)
    real()
    assert os.path.getmtime(build.LIB) == before
    # and a changed fingerprint (what a source edit does) invalidates it
    with open(build.STAMP) as fh:
        stamp = fh.read()
    assert stamp.strip() == build._fingerprint()


def test_peak_probe_is_not_part_of_the_product_abi(lib_path):
    """The bench-only micro-benchmarks live in their own library (libpt_probe.so), not in libpt.so or include/pt.h."""
    from paper_1906_10598_b200 import build
    assert "pt_peak_probe" not in _declared_symbols()
    lib = C.CDLL(lib_path)
    assert not hasattr(lib, "pt_peak_probe") and not hasattr(lib, "pt_bench_peak_probe")
    probe = C.CDLL(build.build_probe())
    assert hasattr(probe, "pt_bench_peak_probe")


def test_header_documents_every_status_bit_and_the_async_contract():
    with open(os.path.join(ROOT, "include", "pt.h")) as fh:
        text = fh.read()
    for bit in ("bit0 (1)", "bit1 (2)", "bit2 (4)", "bit3 (8)", "bit4 (16)"):
        assert bit in text, bit
    assert "never synchronise the device or the stream" in text
    # no non-_host entry point may say that it synchronises
    for m in re.finditer(r"/\*(.*?)\*/\s*(?:typedef struct \{.*?\} \w+;\s*)?PT_API[^;]*?\b(pt_\w+)\s*\(", text, re.S):
        doc, name = m.group(1), m.group(2)
        if not name.endswith("_host") and not name.endswith("_host_q"):
            assert "synchronises `stream`" not in doc, name


def test_refit_workspace_query_and_validation_need_no_gpu(lib_path):
    from paper_1906_10598_b200 import pt
    L = pt.lib()
    cfg = pt.make_config(D=5, NP=128, generations=10, t0=-0.5)
    n = L.pt_refit_doubtful_workspace_bytes(3600, 16000, C.byref(cfg))
    # per_block [B][10] f64 + total phase + flags + list + the device counter, each rounded to 256 bytes
    assert n >= 3600 * (80 + 8 + 4 + 4) + 4 and n % 256 == 0
    dummy = C.c_void_p(256)
    bad = pt.make_retry_config(phi_tol=-1.0, F_tol=1.0)
    assert L.pt_refit_doubtful(dummy, 4, 1000, 1000.0, dummy, dummy, None, C.byref(cfg), C.byref(bad), dummy, dummy, dummy, dummy,
                               dummy, n, None) == -1
    ok = pt.make_retry_config(phi_tol=1.0, F_tol=1.0)
    assert L.pt_refit_doubtful(dummy, 4, 1000, 1000.0, dummy, dummy, None, C.byref(cfg), C.byref(ok), dummy, dummy, dummy, dummy,
                               dummy, 16, None) == -2          # workspace too small


def test_plan_and_error_state_are_thread_safe(lib_path):
    """Per-device state of the library is mutex-guarded and the error string is per thread: hammer the plan query from threads."""
    import threading
    from paper_1906_10598_b200 import pt
    pt.lib()
    errs = []

    def work(k):
        try:
            for _ in range(200):
                cfg = pt.make_config(D=5 + (k & 1), NP=64 * (1 + k % 3), generations=10, t0=-0.5)
                plan = pt.pt_fit_blocks_plan(100 + k, 4096, cfg)
                assert plan["threads"] % 32 == 0
        except Exception as exc:      # pragma: no cover
            errs.append(exc)

    ts = [threading.Thread(target=work, args=(k,)) for k in range(8)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    assert not errs
