"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads, exports every symbol that
include/sail.h declares, validates arguments on the host and refuses to run without a CUDA device
(no CPU fallback).  No compute calls here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1609_07936_b200 import build, binding
    build.build(defines=())
    return binding.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sail.h")).read()
    return sorted(set(re.findall(r"SAIL_API[^;(]*?\b(sail_\w+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    from paper_1609_07936_b200 import binding
    names = _declared_symbols()
    assert len(names) >= 15
    assert sorted(binding.EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), n


def test_workspace_bytes_is_monotone(lib):
    a = lib.sail_workspace_bytes(256, 100, 4096)
    b = lib.sail_workspace_bytes(256, 100, 8192)
    assert 0 < a < b
    assert a >= 4096 * (256 + 100) * 8
    assert lib.sail_workspace_bytes(1, 100, 4096) == 0


def test_create_validates_arguments_before_touching_the_device(lib):
    from paper_1609_07936_b200 import binding
    omega = np.arange(16) * 0.5
    tau = np.arange(8) * 0.1
    F = np.ones(8)
    cfg = binding.sail_config()
    cfg.max_walkers = 4
    h = C.c_void_p()

    def create(om, ta, f, sg=None, n_om=None, n_ta=None):
        return lib.sail_create(C.byref(h), om.ctypes.data, n_om or om.size, ta.ctypes.data, n_ta or ta.size,
                               f.ctypes.data, sg.ctypes.data if sg is not None else None, C.byref(cfg))

    bad = omega.copy(); bad[5] += 1e-6
    assert create(bad, tau, F) == binding.SAIL_ERR_GRID and h.value is None
    assert b"omega" in lib.sail_last_error(None)
    badt = tau.copy(); badt[3] *= 1.01
    assert create(omega, badt, F) == binding.SAIL_ERR_GRID
    assert create(omega[::-1].copy(), tau, F) == binding.SAIL_ERR_GRID
    assert create(omega, tau, F, n_om=1) == binding.SAIL_ERR_ARG
    assert create(omega, np.arange(600) * 0.01, np.ones(600)) == binding.SAIL_ERR_ARG      # n_tau > 512
    assert create(omega, tau, F, sg=np.zeros(8)) == binding.SAIL_ERR_ARG                   # sigma must be > 0
    assert lib.sail_create(None, None, 0, None, 0, None, None, None) == binding.SAIL_ERR_ARG


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1609_07936_b200 import binding
    omega = np.arange(16) * 0.5
    tau = np.arange(8) * 0.1
    F = np.ones(8)
    cfg = binding.sail_config()
    cfg.max_walkers = 4
    h = C.c_void_p()
    rc = lib.sail_create(C.byref(h), omega.ctypes.data, 16, tau.ctypes.data, 8, F.ctypes.data, None, C.byref(cfg))
    assert rc == binding.SAIL_ERR_CUDA and h.value is None
    assert b"no CPU fallback" in lib.sail_last_error(None)
    with pytest.raises(RuntimeError):
        binding.Sail(omega, tau, F, max_walkers=4)
    out = C.c_double()
    assert lib.sail_measure_fp64_peak(0, None, C.byref(out)) == binding.SAIL_ERR_CUDA
    buf = (C.c_double * 16)()
    lib.sail_microbench.argtypes = [C.c_int32, C.c_void_p, C.POINTER(C.c_double), C.c_int32]
    assert lib.sail_microbench(0, None, buf, 16) == binding.SAIL_ERR_CUDA
    assert lib.sail_microbench(0, None, buf, 3) == binding.SAIL_ERR_ARG          # array too short
    assert lib.sail_microbench(0, None, None, 16) == binding.SAIL_ERR_ARG
    lib.sail_smooth.argtypes = [C.c_void_p, C.c_double]
    assert lib.sail_smooth(None, 0.02) == binding.SAIL_ERR_ARG
    assert lib.sail_destroy(None) == 0


def test_product_does_not_import_the_oracle():
    """The CUDA package must not import, read or link anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1609_07936_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, re.M), f
                assert "sail_oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "sail_oracle.c")).read()
    assert "import paper_1609_07936_b200" not in otext and "from paper_1609_07936_b200" not in otext
    assert "sail.h" not in otext.replace("include/sail.h", "")


def test_header_is_plain_c(tmp_path):
    """include/sail.h must compile as C99 (the boundary is a C ABI: no C++ or torch types in the signatures)."""
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "sail.h"\nint main(void) { sail_anneal_params p; sail_selfcool_params q; sail_branch_info i;\n'
                   '  (void)p; (void)q; (void)i; return SAIL_MICROBENCH_N; }\n')
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-fsyntax-only", "-I", os.path.join(ROOT, "include"), str(src)],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
