"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/eagle_verify.h declares; the binding mirrors them; calls fail loudly without a device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_18502_b200 import build, load_library
    build.build()
    return load_library()


def _declared():
    src = open(os.path.join(ROOT, "include", "eagle_verify.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ev_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    from paper_2606_18502_b200 import SIGNATURES
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(SIGNATURES) == names          # binding mirrors the header, name for name


def test_no_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2606_18502_b200.binding import ev_config
    cfg = ev_config(2, 256, 4, 2, 64, 688, 1024, 1e-5, 1e4, 16, 0, 1, 8, 256)
    h = C.c_void_p()
    rc = lib.ev_model_create(C.byref(cfg), C.byref(h))
    assert rc == -4 and b"CUDA" in lib.ev_last_error()          # EV_ECUDA, no silent fallback


def test_argument_validation_precedes_device_use(lib):
    from paper_2606_18502_b200.binding import ev_config
    h = C.c_void_p()
    assert lib.ev_model_create(None, C.byref(h)) == -1
    bad = ev_config(2, 256, 4, 3, 64, 688, 1024, 1e-5, 1e4, 16, 0, 1, 8, 256)       # 4 q heads / 3 kv heads
    assert lib.ev_model_create(C.byref(bad), C.byref(h)) == -1 and b"multiple" in lib.ev_last_error()
    bad = ev_config(2, 256, 4, 2, 96, 688, 1024, 1e-5, 1e4, 16, 0, 1, 8, 256)       # head_dim 96
    assert lib.ev_model_create(C.byref(bad), C.byref(h)) == -1
    bad = ev_config(2, 256, 4, 2, 64, 688, 1024, 1e-5, 1e4, 16, 0, 1, 65, 256)      # T > 64
    assert lib.ev_model_create(C.byref(bad), C.byref(h)) == -1
    assert lib.ev_verify(None, None, None, None, None) == -1
    assert lib.ev_model_destroy(None) == 0 and lib.ev_cache_destroy(None) == 0


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_18502_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("never imports oracle/", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2606_18502_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "paper_2606_18502_b200/", "")
