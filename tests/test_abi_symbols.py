"""The C-ABI library builds here (nvcc cross-compiles for sm_100a), loads, and exports every symbol that
include/wcsim.h declares.  No compute call is made: there is no GPU in this container."""
import ctypes
import os
import re
import shutil

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "wcsim.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(wcsim_[a-z_0-9]+)\s*\(", src)))


@pytest.mark.skipif(shutil.which("nvcc") is None, reason="nvcc not on PATH")
def test_library_exports_every_declared_symbol():
    from paper_2203_02479_b200 import binding, build
    path = build.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), "libwcsim.so does not export %s" % n
    assert sorted(binding.SYMBOLS) == names, "binding.SYMBOLS and include/wcsim.h disagree"


@pytest.mark.skipif(shutil.which("nvcc") is None, reason="nvcc not on PATH")
def test_argument_errors_need_no_device():
    from paper_2203_02479_b200 import binding
    L = binding.lib()
    assert L.wcsim_strerror(0) == b"ok"
    assert L.wcsim_plan_destroy(None) == binding.WCSIM_OK
    assert L.wcsim_convolve(None) == binding.WCSIM_EINVAL
    h = ctypes.c_void_p(123)
    # even response width is rejected before any CUDA call
    import numpy as np
    r = np.zeros((4, 8), dtype=np.float32)
    st = L.wcsim_plan_create(ctypes.byref(h), 8, 32, r.ctypes.data_as(ctypes.c_void_p), 4, 8, binding.wcsim_pad(0, 0),
                             3.0, 0, None)
    assert st == binding.WCSIM_EINVAL and h.value is None
    assert b"sm_100a" in L.wcsim_version()
    # the no-allocation entry point refuses a grid beyond its built-in scratch before it touches the device
    st = L.wcsim_raster_scatter_noalloc(1024, 1024, None, 1, 0, 0, 0, 3.0, ctypes.c_void_p(256), None)
    assert st == binding.WCSIM_ETOOBIG and b"WCSIM_NOALLOC_MAX_BINS" in L.wcsim_strerror(st)
    assert L.wcsim_raster_scatter_noalloc(64, 512, None, 1, 0, 0, 0, 3.0, None, None) == binding.WCSIM_EINVAL


def test_binding_imports_nothing_from_the_oracle():
    for f in ("binding.py", "build.py", "synth.py", "__init__.py"):
        src = open(os.path.join(ROOT, "paper_2203_02479_b200", f)).read()
        assert "import oracle" not in src and "from oracle" not in src
    for f in os.listdir(os.path.join(ROOT, "paper_2203_02479_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_2203_02479_b200", "csrc", f)).read().lower().replace(
            "the oracle", "")
