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


def test_product_path_has_no_oracle_import():
    """The package must not import, read or run anything under oracle/ (the oracle is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_1906_10598_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, f)) as fh:
                    text = fh.read()
                assert "import oracle" not in text and "from oracle" not in text and "pt_oracle" not in text, f
