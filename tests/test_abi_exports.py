"""The C-ABI library builds, loads on a CPU-only box and exports every symbol include/spd.h
declares; host-side logic (width-set generators, argument checks) works without a GPU, and
compute entry points fail loudly instead of falling back to the CPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def spd():
    import paper_1910_08324_b200 as spd
    spd.build()
    return spd


def declared_functions():
    text = open(os.path.join(ROOT, "include", "spd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(spd_[a-z_]+)\s*\(", text)))


def test_header_and_binding_list_the_same_symbols(spd):
    assert declared_functions() == sorted(spd.EXPORTS)


def test_library_exports_every_declared_symbol(spd):
    lib = ctypes.CDLL(spd.LIB_PATH)
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} is declared in include/spd.h but not exported"
    assert spd.spd_version() == 200


def test_library_is_built_for_sm_100a_only(spd):
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", spd.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_width_set_generators_match_paper_examples(spd, paper_pins):
    """Pins P3 through the product's own generator: eq. (14) example PAPER.md:201 and Table 1
    PAPER.md:380-387 (host logic only, no GPU)."""
    assert list(spd.spd_width_set_generate("BOXDIT", 4, 12)) == [1, 2, 3, 4, 6, 8, 10, 12]
    ig = {d: [int(v) for v in spd.spd_width_set_generate("IGRID", d, 31) if v >= 16] for d in (1, 2, 3)}
    assert ig[1] == [16, 24]
    assert ig[2] == [16, 20, 24, 28]
    assert ig[3] == list(range(16, 32, 2))
    assert list(spd.spd_width_set_generate("POW2", 0, 8192)) == [1 << k for k in range(14)]
    assert int(spd.spd_width_set_generate("BOXDIT", 8, 8192)[-1]) == 8184  # footnote 9
    from oracle import formulas
    for kind, param, mw in [("ALL", 0, 64), ("POW2", 0, 32768), ("BOXDIT", 16, 8192), ("BOXDIT", 32, 8192),
                            ("IGRID", 1, 8192), ("IGRID", 2, 16384), ("IGRID", 3, 32768),
                            ("GEOMETRIC", 1800, 8192)]:
        assert list(spd.spd_width_set_generate(kind, param, mw)) == formulas.width_set(kind, param, mw)


def test_separation_generator_matches_formula_module_and_paper_example(spd):
    """Host logic of spd_separation_generate (no device needed): PAPER.md:201 (L_max = 4: widths
    1..4 at every point, 6..12 at every second point), Alg. 3 (width 2^i every 2^i), P layers."""
    from oracle import formulas as F
    w = spd.spd_width_set_generate("BOXDIT", 4, 28)
    assert list(spd.spd_separation_generate("BOXDIT", 4, w)) == [1, 1, 1, 1, 2, 2, 2, 2, 4, 4, 4, 4]
    for l_max in (8, 16, 32):
        w = spd.spd_width_set_generate("BOXDIT", l_max, 8192)
        sep = F.boxdit_separation(l_max)
        assert list(spd.spd_separation_generate("BOXDIT", l_max, w)) == [sep(int(L)) for L in w]
    w = spd.spd_width_set_generate("POW2", 0, 8192)
    assert list(spd.spd_separation_generate("DIT", 0, w)) == list(w)
    for depth, layers in ((1, 4), (2, 8), (3, 16)):
        w = spd.spd_width_set_generate("IGRID", depth, 8192)
        sep = F.igrid_separation(layers)
        assert list(spd.spd_separation_generate("IGRID", layers, w)) == [sep(int(L)) for L in w]
    assert list(spd.spd_separation_generate("EVERY_SAMPLE", 0, [1, 5, 9])) == [1, 1, 1]
    for bad in (("DIT", 0, [3]), ("BOXDIT", 0, [1]), ("IGRID", 3, [4]), (9, 0, [1])):
        with pytest.raises(spd.SpdError):
            spd.spd_separation_generate(*bad)


def test_width_set_generator_errors(spd):
    for kind, param, mw in [(99, 0, 8), ("BOXDIT", 0, 8), ("GEOMETRIC", 1000, 8), ("POW2", 0, 0), ("IGRID", -1, 8)]:
        with pytest.raises(spd.SpdError) as e:
            spd.spd_width_set_generate(kind, param, mw)
        assert e.value.status == -1
    lib = spd.load()
    n = ctypes.c_int32(0)
    buf = np.zeros(2, dtype=np.int32)
    assert lib.spd_width_set_generate(1, 0, 64, buf.ctypes.data, 2, ctypes.byref(n)) == -1
    assert n.value == 7  # size still reported when the capacity is too small


def test_plan_argument_checks_precede_device_checks(spd):
    for args in [(4, 1024, [], 8), (4, 1024, [0, 2], 8), (4, 1024, [16], 8), (4, 64, [1, 2], 128),
                 (0, 1024, [1], 1), (4, 0, [1], 1)]:
        with pytest.raises(spd.SpdError) as e:
            spd.spd_plan_create(*args)
        assert e.value.status == -1, args


def test_no_cpu_fallback_without_a_device(spd):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(spd.SpdError) as e:
        spd.spd_plan_create(4, 1024, [1, 2, 4], 4)
    assert e.value.status == -2
    assert "no CPU fallback" in str(e.value) or "not supported" in str(e.value)


def test_library_reads_no_environment_variable():
    """Kernel choice and work split are plan flags / options (include/spd.h), not process-global state."""
    pkg = os.path.join(ROOT, "paper_1910_08324_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".cu", ".h", ".cuh", ".cpp")):
                assert "getenv" not in open(os.path.join(dirpath, f)).read(), f


def test_spd_destroy_is_a_c_symbol_and_accepts_null(spd):
    lib = spd.load()
    lib.spd_destroy(None)
    lib.spd_plan_destroy(None)
    assert lib.spd_plan_set_option(None, 1, 2) == -1


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1910_08324_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "spd_oracle" not in text and "libspd_oracle" not in text, f
