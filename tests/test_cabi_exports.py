"""The C-ABI library builds here (nvcc cross-compiles sm_100a without a GPU), loads, and exports every
symbol include/gbfit.h declares.  No compute call is made (no GPU in this container)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2405_04690_b200 import build
    return build.build()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "gbfit.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gb_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for must in ("gb_waveform", "gb_delta_loglike", "gb_residual_update", "gb_create", "gb_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    names = declared_functions()
    assert len(names) >= 13
    for n in names:
        assert hasattr(L, n), f"libgbfit.so does not export {n}"


def test_binding_lists_the_same_names(libpath):
    from paper_2405_04690_b200 import gbfit
    assert sorted(gbfit.EXPORTS) == declared_functions()


def test_calls_without_gpu_fail_with_status_not_crash(libpath):
    """No device here: gb_create must return an error code and leave a readable message."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2405_04690_b200 import gbfit
    L = gbfit.lib()
    assert gbfit.version().startswith("gbfit-b200")
    cfg = gbfit.GbConfig()
    L.gb_default_config(ctypes.byref(cfg))
    assert cfg.Tobs == 31457280.0 and cfg.dt == 5.0 and cfg.armlength == 2.5e9
    h = ctypes.c_void_p()
    rc = L.gb_create(ctypes.byref(cfg), ctypes.byref(h))
    assert rc == gbfit.GB_ERR_CUDA
    assert h.value is not None and len(L.gb_last_error(h)) > 0
    L.gb_destroy(h)
    assert L.gb_create(None, ctypes.byref(h)) == gbfit.GB_ERR_INVALID
    assert L.gb_scratch_bytes(None) == 0 and L.gb_launch_count(None) == 0
    with pytest.raises(gbfit.GbError):
        gbfit.Context(0)


def test_product_package_never_touches_the_oracle():
    """The product path may not import, link or read anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2405_04690_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "gb_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2405_04690_b200" not in txt.replace("(paper_2405_04690_b200/)", ""), f
            assert "gbfit.h" not in txt and "csrc" not in txt, f
