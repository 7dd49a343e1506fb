"""CPU-side checks of the boundary (-m "not gpu"): the C-ABI library builds, loads and exports
every symbol include/cavmag.h declares; argument validation that needs no device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2603_03706_b200 import build
    return build.build()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "cavmag.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cav_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for need in ("cav_create", "cav_set_modes", "cav_run", "cav_get_m", "cav_get_a", "cav_set_m", "cav_set_a",
                 "cav_destroy", "cav_get_stats", "cav_set_trace", "cav_get_trace"):
        assert need in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = C.CDLL(lib_path)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/cavmag.h but not exported"


def test_binding_covers_every_declared_symbol(lib_path):
    from paper_2603_03706_b200 import api
    assert sorted(api.EXPORTS) == _declared_symbols()
    for name in api.EXPORTS:
        assert callable(getattr(api, name))


def test_strerror_and_version(lib_path):
    from paper_2603_03706_b200 import api
    assert api.cav_strerror(0) == "ok"
    assert "underflow" in api.cav_strerror(api.CAV_E_DT_UNDERFLOW)
    assert "sm_100a" in api.cav_version()


def test_create_validates_arguments_before_touching_the_device(lib_path):
    from paper_2603_03706_b200 import api
    good = dict(Ms=140e3, Aex=3.7e-12, alpha=1e-3, gamma=1.76e11, B0=(0, 0, 0.1))
    with pytest.raises(api.CavError) as e:
        api.cav_create((0, 8, 8, 5e-9, 5e-9, 5e-9), good)
    assert e.value.status == api.CAV_E_ARG
    with pytest.raises(api.CavError) as e:
        api.cav_create((8, 8, 8, 5e-9, 5e-9, 5e-9), dict(good, n_sub=3))
    assert e.value.status == api.CAV_E_ARG
    with pytest.raises(api.CavError) as e:
        api.cav_create((8, 8, 8, 5e-9, 5e-9, 5e-9), dict(good, Ms=0.0))
    assert e.value.status == api.CAV_E_ARG


def test_binding_refuses_wrong_dtype_or_size(lib_path):
    """The C ABI takes untyped pointers: the binding checks element type and count of every cell-field buffer
    against the handle's precision and shape before the library touches it."""
    import numpy as np
    from paper_2603_03706_b200 import api
    h = 0xDEAD                                   # no device needed: the check runs before the library call
    api._HANDLES[h] = (np.float32, 2, 4 * 3 * 2, 1)
    try:
        ok = np.zeros((2, 3, 2, 3, 4), dtype=np.float32)
        assert api._ptr(ok, *api._field_spec(h))[0] == ok.ctypes.data
        with pytest.raises(ValueError, match="dtype"):
            api.cav_set_m(h, ok.astype(np.float64))
        with pytest.raises(ValueError, match="elements"):
            api.cav_get_m(h, np.zeros((1, 3, 2, 3, 4), dtype=np.float32))
        with pytest.raises(ValueError, match="elements"):
            api.cav_set_modes(h, np.zeros((3, 2, 3, 4), dtype=np.float32), [1.0, 2.0], [0, 0], [0, 0])
        with pytest.raises(ValueError, match="contiguous"):
            api.cav_set_m(h, np.zeros((2, 3, 2, 3, 8), dtype=np.float32)[..., ::2])
        import torch
        with pytest.raises(ValueError, match="dtype"):
            api.cav_get_dmdt(h, torch.zeros((2, 3, 2, 3, 4), dtype=torch.float64))
    finally:
        api._HANDLES.pop(h, None)


def test_no_cpu_fallback_without_device(lib_path):
    """Without a CUDA device the product path fails loudly (CAV_E_UNSUPPORTED); it never
    routes through the oracle."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2603_03706_b200 import api
    with pytest.raises(api.CavError) as e:
        api.cav_create((8, 8, 8, 5e-9, 5e-9, 5e-9), dict(Ms=140e3, Aex=3.7e-12, alpha=1e-3, gamma=1.76e11, B0=(0, 0, 0.1)))
    assert e.value.status == api.CAV_E_UNSUPPORTED


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2603_03706_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("never\nroutes through the oracle", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2603_03706_b200" not in txt and "from paper_2603_03706_b200" not in txt
            assert "cavmag.h" not in txt and "stage_kernel" not in txt
