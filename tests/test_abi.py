"""CPU-side checks of the boundary (no GPU needed): the library builds for sm_100a, loads, exports every
symbol include/lofar_moon.h declares, and its host-only calls validate their arguments."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lofar_moon.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1612_06592_b200 import build, binding
    build.build()
    return binding.load()


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"LOFAR_API[^;(]*?\b(lofar_\w+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for want in ("lofar_plan_create", "lofar_beamform_dedisperse", "lofar_inverse_ppf", "lofar_trigger",
                 "lofar_run_block"):
        assert want in names
    assert len(names) >= 18


def test_library_exports_every_declared_symbol(lib):
    from paper_1612_06592_b200 import binding
    names = declared_symbols()
    assert sorted(binding.EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), n
    # and nothing but the ABI is visible
    out = subprocess.check_output(["nm", "-D", "--defined-only", binding.LIB_PATH], text=True)
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    assert set(names) <= exported
    assert all(s.startswith("lofar_") for s in exported if not s.startswith("_")), exported


def test_header_compiles_as_c99(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "lofar_moon.h"\nint main(void){ lofar_candidate c; return (int)sizeof(c) - 24; }\n')
    exe = tmp_path / "t"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                           str(src), "-o", str(exe)])
    assert subprocess.call([str(exe)]) == 0


def test_library_is_sm100a_with_lineinfo(lib):
    from paper_1612_06592_b200 import binding
    out = subprocess.check_output(["cuobjdump", "-lelf", binding.LIB_PATH], text=True)
    assert "sm_100a" in out


def test_plan_host_side_validation(lib):
    from paper_1612_06592_b200 import binding as b
    h = ctypes.c_void_p()
    assert lib.lofar_plan_create(None, 4, 16, 2, 16, 10.0) == b.LOFAR_E_INVALID
    assert lib.lofar_plan_create(ctypes.byref(h), 0, 16, 2, 16, 10.0) == b.LOFAR_E_INVALID
    assert lib.lofar_plan_create(ctypes.byref(h), 4, 16, 2, 8, 10.0) == b.LOFAR_E_INVALID      # taps != 16
    assert lib.lofar_plan_create(ctypes.byref(h), 4, 513, 2, 16, 10.0) == b.LOFAR_E_SHAPE
    assert lib.lofar_plan_create(ctypes.byref(h), 4, 16, 2, 16, 10.0) == b.LOFAR_OK
    assert lib.lofar_plan_set_band(h, 500, 100e6, 200e6, 1024) == b.LOFAR_E_SHAPE              # 500 + 16 > 512
    assert lib.lofar_plan_set_band(h, 300, 100e6, 200e6, 512) == b.LOFAR_E_INVALID
    assert lib.lofar_plan_set_band(h, 300, 100e6, 200e6, 1024) == b.LOFAR_OK
    assert lib.lofar_plan_set_trials(h, 0, None) == b.LOFAR_E_INVALID
    assert lib.lofar_plan_set_input(h, 2, 64) == b.LOFAR_E_INVALID
    assert lib.lofar_plan_set_input(h, b.LOFAR_CI16, 4096) == b.LOFAR_OK
    assert lib.lofar_plan_set_trigger(h, -1.0, 1, 10) == b.LOFAR_E_INVALID
    assert lib.lofar_plan_set_trigger(h, 5.0, 1, 1000) == b.LOFAR_OK
    n = ctypes.c_size_t()
    assert lib.lofar_plan_workspace_bytes(h, ctypes.byref(n)) == b.LOFAR_OK
    # tables + 2 x history (2 series x 15 x 1024 fp32) + beam-sum scratch (2 x 16 x 4096 float2) + partials
    assert n.value > 2 * 2 * 15 * 1024 * 4 + 2 * 16 * 4096 * 8
    assert lib.lofar_plan_launch_count(h) == 0
    lib.lofar_plan_destroy(h)
    assert b.status_string(b.LOFAR_E_ALIGN).startswith("pointer")


def test_compute_calls_fail_loudly_without_a_gpu(lib):
    """No CPU fallback: on a box without a CUDA device a compute call returns LOFAR_E_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1612_06592_b200 import binding as b
    p = b.Plan(2, 4, 1, 16, 1.0)
    p.set_input(b.LOFAR_CI8, 64)
    X = np.zeros(2 * 2 * 4 * 64 * 2 + 64, dtype=np.int8)
    X = X[(-X.ctypes.data) % 16:]
    Z = np.zeros((1, 4, 64, 2), dtype=np.float32)
    st = p._lib.lofar_beamform_dedisperse(p._h, X.ctypes.data, 64, Z.ctypes.data, None)
    assert st == b.LOFAR_E_CUDA
    p.destroy()


def test_binding_refuses_to_run_without_the_library(monkeypatch, tmp_path):
    from paper_1612_06592_b200 import binding as b
    monkeypatch.setattr(b, "_lib", None)
    monkeypatch.setattr(b, "LIB_PATH", str(tmp_path / "missing.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        b.load()
