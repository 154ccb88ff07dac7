"""The C-ABI library loads and exports every symbol include/jpet.h declares (no compute, CPU only)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "jpet.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(jpet_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_calls_of_the_scope_table():
    syms = declared_symbols()
    for must in ("jpet_sensitivity", "jpet_mlem_iterate", "jpet_reconstruct", "jpet_mlem_begin", "jpet_mlem_accumulate",
                 "jpet_mlem_end", "jpet_count_evals", "jpet_last_error"):
        assert must in syms


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1502_07478_b200 import binding, build

    path = build.build()
    assert os.path.exists(path)
    lib = binding.load()
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/jpet.h but not exported by libjpet.so"
    assert sorted(binding.EXPORTS) == declared_symbols()
    assert lib.jpet_abi_version() == 2


def test_library_is_sm100a_native():
    import subprocess

    from paper_1502_07478_b200 import build

    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump not available")
    assert "sm_100a" in out.stdout


def test_argument_validation_needs_no_gpu():
    """Calls that fail validation return JPET_E_INVAL before touching CUDA."""
    import ctypes

    from paper_1502_07478_b200 import binding

    lib = binding.load()
    g, s, gr = binding.Geometry(450, 500), binding.Sigmas(10, 40), binding.Grid(64, 64, 5.0)
    assert lib.jpet_sensitivity(None, gr, None, None) == binding.JPET_E_INVAL
    assert lib.jpet_sensitivity(g, gr, None, None) == binding.JPET_E_INVAL
    assert b"NULL" in lib.jpet_last_error()
    bad = binding.Grid(400, 64, 5.0)   # |y| reaches 997 mm >= R
    assert lib.jpet_mlem_iterate(None, 0, g, s, bad, None, None, None) == binding.JPET_E_INVAL
    assert b"R" in lib.jpet_last_error()
    assert lib.jpet_mlem_iterate(None, -1, g, s, gr, None, None, None) == binding.JPET_E_INVAL
    assert lib.jpet_mlem_iterate(None, 0, g, binding.Sigmas(0, 40), gr, None, None, None) == binding.JPET_E_INVAL
    assert lib.jpet_mlem_iterate(None, 0, g, binding.Sigmas(300, 40), gr, None, None, None) == binding.JPET_E_INVAL
    assert lib.jpet_mlem_accumulate(None, 0, None) == binding.JPET_E_INVAL   # no begin
    assert lib.jpet_mlem_end(None, None, None) == binding.JPET_E_INVAL
    assert lib.jpet_set_option(b"nonsense", 1) == binding.JPET_E_INVAL
    assert lib.jpet_set_option(b"chunk", -5) == binding.JPET_E_INVAL
    assert lib.jpet_set_a3_coef(ctypes.c_float(float("nan"))) == binding.JPET_E_INVAL
    assert abs(lib.jpet_get_a3_coef() - 2.0) < 1e-7
    assert lib.jpet_set_gamma(ctypes.c_float(float("inf"))) == binding.JPET_E_INVAL
    assert lib.jpet_get_gamma() == 0.0
    # Eq. 12 must stay positive definite: |gamma| <= 0.5 / (sqrt(2) sigma_z sigma_dl), checked against the call's sigmas
    assert lib.jpet_set_gamma(ctypes.c_float(1e-2)) == binding.JPET_OK
    assert lib.jpet_mlem_iterate(None, 0, g, s, gr, None, None, None) == binding.JPET_E_INVAL
    assert b"gamma" in lib.jpet_last_error()
    assert lib.jpet_set_gamma(ctypes.c_float(0.0)) == binding.JPET_OK
    # the calls added in round 2 validate before touching CUDA as well
    assert lib.jpet_set_sigma_z_edge(ctypes.c_float(-0.1)) == binding.JPET_E_INVAL
    assert lib.jpet_set_sigma_z_edge(ctypes.c_float(float("nan"))) == binding.JPET_E_INVAL
    assert lib.jpet_get_sigma_z_edge() == 0.0
    assert lib.jpet_direct_histogram(None, 5, g, gr, None, None, None) == binding.JPET_E_INVAL
    assert lib.jpet_direct_histogram(None, 0, g, gr, None, None, None) == binding.JPET_E_INVAL          # NULL histogram
    prim = (binding.Primitive * 1)(binding.Primitive(0, 0, 0, 10, 10, 0, 0.0))
    assert lib.jpet_generate_events(prim, 1, 0, 0, g, s, 1, None, None) == binding.JPET_E_INVAL            # no positive intensity
    assert lib.jpet_generate_events(prim, 0, 0, 0, g, s, 1, None, None) == binding.JPET_E_INVAL
    assert lib.jpet_mlem_end_peers(None, None, None, 2, None) == binding.JPET_E_INVAL
    assert lib.jpet_ipc_export(None, None) == binding.JPET_E_INVAL
    assert lib.jpet_set_option(b"exact_kernel", 5000) == binding.JPET_E_INVAL
    assert lib.jpet_shape_name(0) == b"small_closed" and lib.jpet_shape_name(99) == b""


def test_product_does_not_reach_into_the_oracle():
    """Neither side imports, includes, links or executes the other (the oracle is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_1502_07478_b200")
    reach = re.compile(r"^\s*(import\s+oracle|from\s+oracle\b|#\s*include\s+.*oracle)|jpet_oracle|libjpet_oracle|jo_[a-z]", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not reach.search(open(os.path.join(dirpath, f)).read()), f
    assert not reach.search(open(os.path.join(ROOT, "include", "jpet.h")).read())
    back = re.compile(r"^\s*(import|from)\s+paper_1502_07478_b200|#\s*include\s+.*(jpet\.h|csrc|mlem_kernels)|libjpet\.so", re.M)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            assert not back.search(open(os.path.join(ROOT, "oracle", f)).read()), f
