"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/dimos.h declares; the binding refuses to run without a CUDA device (no CPU fallback);
the product package never touches oracle/."""
import ctypes
import os
import re

import pytest
import torch

from paper_2503_20541_b200 import binding, build_ext

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "dimos.h")).read()
    return sorted(set(re.findall(r"DIMOS_API\s+[\w\s\*]+?\b(dimos_\w+)\s*\(", text)))


def test_header_declares_the_three_north_star_calls():
    names = declared_symbols()
    for must in ("dimos_nl_build", "dimos_nl_needs_rebuild", "dimos_nonbonded"):
        assert must in names
    assert set(names) == set(binding.EXPORTED_SYMBOLS)


def test_library_builds_and_exports_every_declared_symbol():
    path = build_ext.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/dimos.h but not exported"
    lib.dimos_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.dimos_version()
    lib.dimos_status_string.restype = ctypes.c_char_p
    lib.dimos_status_string.argtypes = [ctypes.c_int]
    assert lib.dimos_status_string(0) == b"DIMOS_OK"
    assert b"DIMOS_EBOX" in lib.dimos_status_string(-2)


def test_built_for_sm_100a_only():
    out = os.popen(f"cuobjdump -lelf {build_ext.build()} 2>/dev/null").read()
    if not out:
        pytest.skip("cuobjdump not available")
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback_without_a_device():
    lib = binding.load_library()
    h = ctypes.c_void_p()
    assert lib.dimos_create(ctypes.byref(h), 0, 0, None) == -5  # DIMOS_ECUDA
    assert not h.value
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.Context(0, "f32")


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2503_20541_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "liboracle" not in text and "dimos_oracle" not in text, f


def test_lj_table_fill_is_eq5_and_matches_the_oracle():
    """dimos_lj_table_fill (host-only entry point, Eq. 5) against the oracle's Lorentz-Berthelot table
    and against the rule written out: sigma_ab arithmetic mean, eps_ab geometric mean, symmetric."""
    import numpy as np

    import oracle

    sigma, eps = [0.315061, 0.0, 0.25, 0.4], [0.6364, 0.0, 0.3, 1.2]
    t = binding.dimos_lj_table_fill(sigma, eps).numpy()
    assert np.allclose(t, oracle.lorentz_berthelot(sigma, eps), rtol=1e-15, atol=0)
    assert t[0, 2, 0] == 0.5 * (0.315061 + 0.25) and t[0, 2, 1] == pytest.approx((0.6364 * 0.3) ** 0.5, rel=1e-15)
    assert np.array_equal(t, t.transpose(1, 0, 2))
    assert t[1, 1, 1] == 0.0 and t[0, 1, 1] == 0.0  # a type with eps = 0 has no LJ partner
    with pytest.raises(binding.DimosError):
        binding.dimos_lj_table_fill([0.3, -1.0], [0.1, 0.1])


def test_binding_structs_match_the_header_layout(tmp_path):
    """The ctypes mirrors of dimos_nb_params and dimos_nl_stats_t have the size and field offsets a C compiler gives the
    structs of include/dimos.h (the header is plain C: it must compile with gcc, too)."""
    import shutil
    import subprocess

    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no C compiler")
    fields_p = [name for name, _ in binding._Params._fields_]
    fields_s = [name for name, _ in binding._Stats._fields_]
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "dimos.h"', "int main(void) {",
             '  printf("%zu\\n", sizeof(dimos_nb_params));']
    lines += [f'  printf("%zu\\n", offsetof(dimos_nb_params, {f}));' for f in fields_p]
    lines += ['  printf("%zu\\n", sizeof(dimos_nl_stats_t));']
    lines += [f'  printf("%zu\\n", offsetof(dimos_nl_stats_t, {f}));' for f in fields_s]
    lines += ["  return 0;", "}"]
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run([gcc, "-std=c99", "-Wall", "-Werror", "-I", build_ext.INCLUDE, str(src), "-o", str(exe)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    want = [ctypes.sizeof(binding._Params)] + [getattr(binding._Params, f).offset for f in fields_p]
    want += [ctypes.sizeof(binding._Stats)] + [getattr(binding._Stats, f).offset for f in fields_s]
    assert got == want
