"""CPU-side checks: the C-ABI library loads and exports every symbol include/cbgmres.h declares, and
the algorithmic-bytes model reproduces the values the paper prints (tests/golden/paper_values.txt)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _golden():
    vals = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_values.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            vals[k.strip()] = v.strip()
    return vals


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2009_12101_b200 import build as b

    lib_path = b.build()
    header = open(os.path.join(ROOT, "include", "cbgmres.h")).read()
    declared = set(re.findall(r"^(?:int|int64_t|const char \*)\s*(cbgmres_[a-z_0-9]+)\(", header, re.M))
    assert len(declared) >= 16
    lib = ctypes.CDLL(lib_path)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in cbgmres.h but not exported"
    from paper_2009_12101_b200 import EXPORTS

    assert set(EXPORTS) == declared


def test_binding_refuses_to_run_without_cuda():
    import torch

    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    from paper_2009_12101_b200 import Solver

    with pytest.raises(RuntimeError, match="no CPU fallback"):
        Solver()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2009_12101_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "liboracle" not in src and "cbgmres_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "cbgmres_oracle.c")).read()
    assert "import paper_2009_12101_b200" not in osrc and "from paper_2009_12101_b200" not in osrc
    assert "cbgmres.h" not in osrc


def test_memop_model_matches_the_paper():
    from paper_2009_12101_b200 import model

    g = _golden()
    s = model.memop_crossover_s(100, float(g["f_int32_over_fp64"]))
    # the paper prints 67 for the solution of m / (s (1+f) + f) = 1, i.e. 66.33 rounded up
    assert abs(s - 66.3333) < 1e-3 and round(s + 0.5) == int(g["memop_crossover_s_m100_f0.5"])
    assert abs(model.memop_ratio_cycle(100, s) - 1.0) < 1e-12
    # asymptotic speedups = ratio of storage widths
    assert model.FORMAT_BYTES["fp64"] / model.FORMAT_BYTES["fp16"] == int(g["asymptote_16bit"])
    assert model.FORMAT_BYTES["fp64"] / model.FORMAT_BYTES["int32"] == int(g["asymptote_32bit"])
    assert len(model.FORMAT_BYTES) == int(g["n_formats"])


def test_bytes_model_against_survey_table():
    from paper_2009_12101_b200 import model

    # C2 fp64: S1 103 MB, S2+S3 at j = 50.5 ~ 832 MB, S4 24 MB
    n, nnz = 1_000_000, 6_940_000
    assert round(model.spmv_bytes(n, nnz) / 1e6) == 103
    s23 = (model.multidot_bytes(n, 50, "fp64") + model.update_bytes(n, 50, "fp64")
           + model.multidot_bytes(n, 51, "fp64") + model.update_bytes(n, 51, "fp64")) / 2
    assert round(s23 / 1e6) == 832
    assert model.store_bytes(n, "fp64") == 24 * n and model.store_bytes(n, "int16") == 18 * n
    assert model.arnoldi_step_bytes(n, nnz, 10, "fp32", reorth=True) - model.arnoldi_step_bytes(n, nnz, 10, "fp32") \
        == model.multidot_bytes(n, 10, "fp32") + model.update_bytes(n, 10, "fp32")


def test_cycle_bytes_model_has_the_papers_asymptotes():
    """the per-cycle speedup of a 32-bit (16-bit) basis approaches a value below 2x (4x) as
    the restart length grows, because the SpMV and the vector traffic do not shrink.  The algorithmic
    bytes model of cyclebench.py must show exactly that."""
    from paper_2009_12101_b200.cyclebench import cycle_bytes

    n, nnz = 1_000_000, 6_940_000
    prev32 = prev16 = 1.0
    for m in (10, 50, 100, 300, 3000):
        r32 = cycle_bytes(n, nnz, m, "fp64", 0.0) / cycle_bytes(n, nnz, m, "fp32", 0.0)
        r16 = cycle_bytes(n, nnz, m, "fp64", 0.0) / cycle_bytes(n, nnz, m, "int16", 0.0)
        assert prev32 < r32 < 2.0 and prev16 < r16 < 4.0 and r16 > r32
        prev32, prev16 = r32, r16
    assert prev32 > 1.98 and prev16 > 3.9
    # re-orthogonalised steps read the basis three times instead of two
    m, B = 100, 4
    extra = cycle_bytes(n, nnz, m, "fp32", 1.0) - cycle_bytes(n, nnz, m, "fp32", 0.0)
    assert extra == sum(j * n * B + 16 * n for j in range(1, m + 1))
    assert cycle_bytes(n, nnz, m, "fp32", 0.0) == cycle_bytes(n, nnz, m, "int32", 0.0)


def test_paper_protocol_matrix_set_uses_known_configs():
    from paper_2009_12101_b200 import paperprotocol
    from workloads import make_config
    from workloads.generators import CONFIG_NAMES

    for label, cfg, kw in paperprotocol.MATRICES + paperprotocol.SMALL:
        assert cfg in CONFIG_NAMES and set(kw) <= {"grid", "n"}
    p = make_config(*paperprotocol.SMALL[0][1:2], **paperprotocol.SMALL[0][2])
    assert p.A.n == 24 ** 3
