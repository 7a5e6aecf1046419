"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol that
include/cbm_trigger.h declares, validates its configuration before touching CUDA, and fails
loudly (no CPU fallback) when there is no device.  No compute calls here."""
import ctypes
import os
import re

import pytest

from paper_1810_11966_b200 import build as B
from paper_1810_11966_b200 import binding as K
from paper_1810_11966_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build_library()
    return K.load_library()


def declared_symbols():
    names = set()
    inc = os.path.join(ROOT, "include")
    for fn in os.listdir(inc):
        if fn.endswith(".h"):
            text = open(os.path.join(inc, fn)).read()
            text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
            names |= set(re.findall(r"\b(cbm_trigger_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_library_exports_every_declared_symbol(lib):
    decl = declared_symbols()
    assert len(decl) >= 9
    for name in decl:
        assert hasattr(lib, name), f"{name} declared in include/ but not exported"
    assert set(decl) == set(K.EXPORTS)


def test_struct_layouts_match_header(lib):
    # sizeof() as the C compiler sees it: compile a probe with gcc against the header
    import subprocess
    import tempfile
    src = '#include "cbm_trigger.h"\n#include <stdio.h>\nint main(){printf("%zu %zu %zu %zu\\n", sizeof(cbm_trigger_config_t), sizeof(cbm_trigger_stats_t), sizeof(cbm_trigger_ubench_t), sizeof(cbm_trigger_msd_params_t));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "p.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "p")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.split()
    assert int(out[0]) == ctypes.sizeof(K.Config)
    assert int(out[1]) == ctypes.sizeof(K.Stats)
    assert int(out[2]) == ctypes.sizeof(K.Ubench)
    assert int(out[3]) == ctypes.sizeof(K.MsdParams)


def test_version(lib):
    assert "sm_100a" in K.cbm_trigger_version()


def _cfg(**kw):
    base = dict(layer_z=list(W.GEOMETRY_4), max_events=100, max_hits=10000)
    base.update(kw)
    return K.make_config(**base)


@pytest.mark.parametrize("mutate,needle", [
    (lambda c: setattr(c, "struct_size", 8), "struct_size"),
    (lambda c: setattr(c, "n_stations", 0), "n_stations"),
    (lambda c: setattr(c, "n_stations", 9), "n_stations"),
    (lambda c: c.layer_z.__setitem__(3, c.layer_z[2]), "increasing"),
    (lambda c: c.layer_z.__setitem__(0, 0), "layer_z"),
    (lambda c: c.layer_z.__setitem__(11, (1 << 23) + 1), "layer_z"),
    (lambda c: setattr(c, "win_in_den", 0), "windows"),
    (lambda c: setattr(c, "win_link_den", 5000), "windows"),
    (lambda c: setattr(c, "win_in_num", 101), "windows"),
    (lambda c: setattr(c, "max_hits_per_layer", 5000), "max_hits_per_layer"),
    (lambda c: setattr(c, "max_hits_per_layer", 0), "max_hits_per_layer"),
    (lambda c: setattr(c, "n_slots", 5), "n_slots"),
    (lambda c: setattr(c, "max_events", 0), "max_events"),
    (lambda c: setattr(c, "max_hits", 1 << 32), "max_hits"),
    # 12 layers: max_events * 12 + 1 one step above CBM_TRIGGER_MAX_INDEX = 2^32 - 8192 (the uint32 block arithmetic of
    # the device scans must not wrap)
    (lambda c: setattr(c, "max_events", 0xFFFFE000 // 12 + 1), "max_events * layers"),
    (lambda c: setattr(c, "tiny_max_layer_hits", 33), "tiny_max_layer_hits"),
])
def test_create_rejects_bad_config_before_cuda(lib, mutate, needle):
    c = _cfg()
    mutate(c)
    with pytest.raises(K.CbmTriggerError) as ei:
        K.cbm_trigger_create(c)
    assert ei.value.code == K.CBM_ERR_INVALID_ARG
    assert needle in str(ei.value)


def test_create_null_arguments(lib):
    h = ctypes.c_void_p()
    assert lib.cbm_trigger_create(None, ctypes.byref(h)) == K.CBM_ERR_INVALID_ARG
    assert lib.cbm_trigger_create(ctypes.byref(_cfg()), None) == K.CBM_ERR_INVALID_ARG
    lib.cbm_trigger_destroy(None)  # allowed


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(K.CbmTriggerError) as ei:
        K.cbm_trigger_create(_cfg())
    assert ei.value.code == K.CBM_ERR_CUDA
    assert "no CPU fallback" in str(ei.value)


def test_missing_library_raises(monkeypatch):
    monkeypatch.setattr(K, "_lib", None)
    monkeypatch.setattr(K, "LIB_PATH", os.path.join(ROOT, "does_not_exist.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        K.load_library()


def test_product_does_not_import_the_oracle():
    # the product path (package + bench's own arm) must never route through oracle/
    pkg = os.path.join(ROOT, "paper_1810_11966_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".c")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), fn
                assert "liboracle" not in text, fn
