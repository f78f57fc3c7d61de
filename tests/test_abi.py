"""CPU-only checks of the C-ABI boundary: the library loads, exports every symbol include/u1gf.h declares, validates
arguments before touching a device and refuses to compute without an sm_100 GPU (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1403_0555_b200 import build, binding as b
    build.build()
    b.lib()
    return b


def _declared_symbols(header="u1gf.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(u1gf_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound(binding):
    declared = _declared_symbols()
    assert len(declared) >= 19
    L = C.CDLL(binding.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/u1gf.h but not exported by libu1gf.so"
    assert declared == binding.exported_symbols(), "binding._SIGNATURES must list exactly the header's symbols"
    assert binding.lib().u1gf_abi_version() == 3
    # the method's header carries no measurement or debug entry points; those live in include/u1gf_measure.h
    assert not [n for n in declared if "measure" in n or n.startswith("u1gf_last_") and n != "u1gf_last_error"]


def test_measure_header_symbols(binding):
    declared = _declared_symbols("u1gf_measure.h")
    assert declared == binding.measure_symbols()
    main, meas = C.CDLL(binding.LIB_PATH), C.CDLL(binding.MEASURE_LIB_PATH)
    for name in declared:
        where = main if name == "u1gf_last_launch_count" else meas
        assert hasattr(where, name), f"{name} declared in include/u1gf_measure.h but not exported"
    for name in declared:
        if name != "u1gf_last_launch_count":
            assert not hasattr(main, name), f"{name}: measurement code inside the method library"


def test_argument_validation_needs_no_device(binding):
    L = binding.lib()
    h = C.c_void_p()
    ext = np.array([4, 4], dtype=np.int32)
    th = np.zeros(32)
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    assert L.u1gf_create_orbit(0, p(ext), p(th), C.byref(h)) == -1 and b"outside 1..4" in L.u1gf_last_error()
    assert L.u1gf_create_orbit(5, p(ext), p(th), C.byref(h)) == -1
    bad = np.array([4, 1], dtype=np.int32)
    assert L.u1gf_create_orbit(2, p(bad), p(th), C.byref(h)) == -1 and b"extent[1]" in L.u1gf_last_error()
    big = np.array([128, 128], dtype=np.int32)
    assert L.u1gf_create_orbit(2, p(big), p(th), C.byref(h)) == -1 and b"volume" in L.u1gf_last_error()
    thn = th.copy(); thn[3] = np.nan
    assert L.u1gf_create_orbit(2, p(ext), p(thn), C.byref(h)) == -1 and b"not finite" in L.u1gf_last_error()
    assert L.u1gf_create_orbit(2, None, p(th), C.byref(h)) == -1
    assert L.u1gf_relax_batch(None, 1, 0, 4, None, 1.7, 1e-13, 100, 1, None, None, None, None, None, None, 0, None) == -1
    assert L.u1gf_check_fp(None, 1, None, None, 1e-8, None, None, None, None, None) == -1
    assert L.u1gf_count_copies(1 << 31, None, None, None, 1e-10, 1e-4, None, None, None, None, None, 0, None, 0, None) == -1
    assert L.u1gf_destroy_orbit(None) == 0
    assert L.u1gf_orbit_volume(None) == 0 and L.u1gf_orbit_dim(None) == 0
    assert L.u1gf_count_workspace_bytes(1000) > 1000 * 40


def test_no_cpu_fallback(binding):
    """Without a CUDA device every compute entry point fails loudly with U1GF_ENODEV."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.U1gfError) as e:
        binding.Orbit((4, 4), np.zeros(32))
    assert e.value.code == -2 and "no CPU fallback" in str(e.value)
    with pytest.raises(binding.U1gfError) as e:
        binding.count_copies_host(np.zeros(4), np.zeros((4, 4)), np.zeros(4, np.uint8))
    assert e.value.code == -2


def test_product_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the package may import or load it."""
    pkg = os.path.join(ROOT, "paper_1403_0555_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "u1gf_oracle" not in src, f
