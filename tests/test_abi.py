"""The C-ABI boundary without a GPU: the library loads, exports every symbol include/mppi.h
declares, the header is plain C and agrees with the Python struct mirror, parameters are
validated, and there is no CPU fallback (mppi_create fails loudly without a device)."""
import ctypes as C
import re
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def B():
    from paper_2509_14726_b200 import build
    build.build()
    from paper_2509_14726_b200 import binding
    return binding


def _declared():
    text = (ROOT / "include" / "mppi.h").read_text()
    return sorted(set(re.findall(r"^MPPI_API [\w\s\*]+?\b(mppi_\w+)\(", text, flags=re.M)))


def test_every_declared_symbol_is_exported(B):
    names = _declared()
    assert len(names) >= 17
    assert sorted(B.EXPORTS) == names
    out = subprocess.run(["nm", "-D", "--defined-only", str(B.LIB_PATH)], capture_output=True, text=True).stdout
    exported = set(re.findall(r" T (mppi_\w+)", out))
    assert set(names) <= exported
    # nothing but the C ABI leaks out of the library
    assert all(n.startswith("mppi_") for n in re.findall(r" T (\w+)", out))


def test_header_is_plain_c_and_matches_python_mirror(B, tmp_path):
    src = tmp_path / "t.c"
    fields = [f for f, _ in B.MppiParams._fields_]
    cf = ["lambda" if f == "lambda_" else f for f in fields]
    body = "".join(f'printf("%zu\\n", offsetof(mppi_params, {f}));\n' for f in cf)
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "mppi.h"\nint main(void){\n'
                   'printf("%zu %zu\\n", sizeof(mppi_params), sizeof(mppi_info));\n' + body + "return 0;}\n")
    exe = tmp_path / "t"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", f"-I{ROOT / 'include'}", str(src), "-o", str(exe)],
                   check=True)
    lines = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split("\n")
    sp, si = (int(v) for v in lines[0].split())
    assert sp == C.sizeof(B.MppiParams) and si == C.sizeof(B.MppiInfo)
    for f, off in zip(fields, lines[1:]):
        assert getattr(B.MppiParams, f).offset == int(off), f


def test_default_params_are_config0(B):
    p = B.default_params()
    assert p.struct_size == C.sizeof(B.MppiParams)
    assert (p.K, p.N, p.B, p.objective) == (256, 20, 1, 0)
    assert p.mass == pytest.approx(0.85) and p.T_max == 7.0 and p.window == 16 and p.lambda_ == 1.0
    assert B.lib.mppi_default_params(None) == -1


@pytest.mark.parametrize("field,value", [("K", 0), ("K", 100), ("N", 0), ("N", 257), ("B", 0),
                                         ("objective", 5), ("objective", 4), ("q_near", -1.0), ("r_near", float("nan")), ("dt", 0.0), ("lambda_", 0.0), ("lambda_", -1.0),
                                         ("sigma", -0.1), ("mass", 0.0), ("Jz", -1.0), ("T_min", 8.0),
                                         ("window", 0), ("window", 65), ("pipeline", 2),
                                         ("block_threads", 48), ("block_threads", 512), ("dt", float("nan"))])
def test_bad_parameters_are_rejected(B, field, value):
    p = B.default_params()
    setattr(p, field, value)
    h = C.c_void_p()
    assert B.lib.mppi_create(C.byref(p), C.byref(h)) == -2          # MPPI_E_PARAM
    assert not h.value
    assert len(B.lib.mppi_last_error(None)) > 0


def test_struct_size_versions_the_abi(B):
    p = B.default_params()
    p.struct_size -= 4
    h = C.c_void_p()
    assert B.lib.mppi_create(C.byref(p), C.byref(h)) == -2
    assert B.lib.mppi_create(None, C.byref(h)) == -1


def test_error_strings(B):
    texts = {B.lib.mppi_error_string(c).decode() for c in range(-8, 1)}
    assert len(texts) == 9 and "ok" in texts
    assert B.lib.mppi_destroy(None) == 0


def test_no_cpu_fallback(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(B.MppiError) as e:
        B.Mppi()
    assert e.value.status == -6                                    # MPPI_E_CUDA, loudly
    t = C.c_double(); f = C.c_double()
    assert B.lib.mppi_measure_fma_peak(1, C.byref(t), C.byref(f)) != 0


def test_product_does_not_touch_the_oracle():
    # the package never imports, links, includes or reads oracle/ (and the oracle never the package)
    bad = re.compile(r"(^\s*(from|import)\s+oracle\b|#include\s+[<\"].*oracle|mppi_oracle|[\"']oracle[\"/'])", re.M)
    for f in (ROOT / "paper_2509_14726_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".cuh", ".h"):
            assert not bad.search(f.read_text()), f
    for f in list((ROOT / "oracle").glob("*.py")) + [ROOT / "oracle" / "mppi_oracle.c"]:
        text = f.read_text()
        assert not re.search(r"(^\s*(from|import)\s+paper_2509_14726_b200|#include\s+[<\"].*(csrc|mppi\.h|cuh))", text, re.M), f
