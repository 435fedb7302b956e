"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads,
and exports every function include/hk.h declares; the binding lists the same
names; host-side argument validation that needs no device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hk.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hk_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2101_02005_b200 import build
    return C.CDLL(build.build())


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ("hk_create", "hk_set_conditions", "hk_compute", "hk_destroy", "hk_workspace_bytes",
                 "hk_set_workspace", "hk_get_stats", "hk_get_extents", "hk_compute_host"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared():
        assert hasattr(lib, name), f"libhk.so does not export {name}"


def test_binding_lists_the_same_symbols(lib):
    from paper_2101_02005_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_library_is_sm100a_native():
    """The fat binary holds sm_100a SASS (cuobjdump), i.e. it was not built for a generic arch."""
    import shutil
    import subprocess
    from paper_2101_02005_b200 import build
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not on PATH")
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_host_side_argument_validation(lib):
    """Checks that happen before any CUDA call (include/hk.h 'Errors')."""
    lib.hk_create.argtypes = [C.c_double, C.c_double, C.c_double, C.POINTER(C.c_void_p)]
    lib.hk_strerror.restype = C.c_char_p
    ctx = C.c_void_p()
    EINVAL = -1
    assert lib.hk_create(0.0, 10.0, 0.0, C.byref(ctx)) == EINVAL          # dnu <= 0
    assert lib.hk_create(10.0, 0.0, 0.1, C.byref(ctx)) == EINVAL          # numax <= numin
    assert lib.hk_create(0.0, float("nan"), 0.1, C.byref(ctx)) == EINVAL
    assert lib.hk_create(0.0, 1e12, 1e-3, C.byref(ctx)) == EINVAL         # N >= 2^31
    assert lib.hk_create(0.0, 10.0, 0.1, None) == EINVAL
    assert ctx.value is None
    lib.hk_set_conditions.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double]
    assert lib.hk_set_conditions(None, 300.0, 1.0, 18.0, 1.0) == EINVAL
    assert lib.hk_strerror(0) == b"ok"
    assert b"workspace" in lib.hk_strerror(-3)
    assert lib.hk_destroy(None) == 0
