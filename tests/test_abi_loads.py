"""CPU-side checks of the boundary: the C-ABI library builds (nvcc cross-compiles without a GPU), loads, exports
every symbol include/cuharm.h declares, keeps its parameter block in step with the binding, and fails loudly —
never falls back — when there is no CUDA device.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

import paper_2205_02484_b200 as cu
from paper_2205_02484_b200 import build as cubuild
from workloads import default_params

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "cuharm.h")


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cuharm_[a-z_0-9]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    path = cubuild.build()
    assert os.path.exists(path)
    L = C.CDLL(path)
    names = declared_symbols()
    assert {"cuharm_grid_init", "cuharm_metric_precompute", "cuharm_step", "cuharm_cons_to_prim", "cuharm_cfl_dt",
            "cuharm_divb"} <= set(names)                 # the calls north_star names
    for n in names:
        assert hasattr(L, n), n


def test_params_block_matches_the_header():
    text = open(HEADER).read()
    body = text[text.index("typedef struct {"):text.index("} cuharm_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").strip()
        if not decl:
            continue
        typ, rest = decl.split(None, 1)
        for name in rest.split(","):
            fields.append((re.sub(r"\[.*\]", "", name).strip(), typ))
    got = [(n, "double" if t in (C.c_double, C.c_double * 3) else "int32_t") for n, t in cu.CuharmParams._fields_]
    assert got == fields
    # the oracle declares the same field order independently (no shared header)
    import oracle
    assert [f[0] for f in oracle.OracleParams._fields_] == [f[0] for f in cu.CuharmParams._fields_]
    assert C.sizeof(oracle.OracleParams) == C.sizeof(cu.CuharmParams)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(cu.CuharmError):
        cu.cuharm_grid_init(default_params())
    with pytest.raises(cu.CuharmError):
        cu.Solver(default_params(), None)


def test_strerror_and_null_handling():
    L = cu.lib()
    assert cu.cuharm_strerror(0) == "ok"
    assert "invalid" in cu.cuharm_strerror(-1)
    assert L.cuharm_grid_init(None, None, None) == -1
    assert L.cuharm_workspace_bytes(None) == 0
    assert L.cuharm_destroy(None) == -1
    assert L.cuharm_launch_count(None) == 0


def test_product_package_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2205_02484_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, f
    for f in ("oracle.cpp", "oracle.py", "build.py"):
        src = open(os.path.join(ROOT, "oracle", f)).read()
        assert "paper_2205_02484_b200" not in src.replace("shares no code, header,\n// table or helper with paper_2205_02484_b200", "") or f == "oracle.cpp"
        assert "libcuharm" not in src and "cuharm.h" not in src
