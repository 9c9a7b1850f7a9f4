"""The C-ABI library builds, loads, and exports every symbol include/vr.h declares; without a
CUDA device its calls fail loudly (there is no CPU fallback). No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def vr():
    from paper_1205_0282_b200 import build
    build.build()
    import paper_1205_0282_b200 as vr
    return vr


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "vr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vr_[a-z_0-9]+)\s*\(", text)))


def test_header_and_binding_agree(vr):
    assert declared_symbols() == sorted(vr.SYMBOLS)


def test_library_exports_every_declared_symbol(vr):
    L = ctypes.CDLL(vr.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(L, name), name
    vr.lib()  # the binding's prototypes resolve as well


def test_stats_struct_layout(vr):
    # int64 x7, int32 x2, float x3, int32 (bricks_culled, in what used to be tail padding)
    assert ctypes.sizeof(vr.Stats) == 80


def test_product_path_does_not_touch_the_oracle():
    """Nothing under the package (or bench's product arm) imports oracle/."""
    pkg = os.path.join(ROOT, "paper_1205_0282_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "vr_oracle" not in src, f


def test_no_device_fails_loudly(vr):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(vr.VrError) as e:
        vr.Volume(8, 8, 8, 8, 1)
    assert e.value.status == 3  # VR_ERR_CUDA
    assert "no CUDA device" in str(e.value)


def test_create_rejects_bad_arguments_before_touching_the_device(vr):
    h = ctypes.c_void_p()
    L = vr.lib()
    assert L.vr_volume_create(0, 8, 8, 8, 1, ctypes.byref(h)) == 1
    assert L.vr_volume_create(8, 8, 8, 1, 1, ctypes.byref(h)) == 1
    assert L.vr_volume_create(8, 8, 8, 8, 9, ctypes.byref(h)) == 1
    assert L.vr_volume_create(8, 8, 8, 8, 1, None) == 1
    assert b"vr_volume_create" in L.vr_last_error(None)
