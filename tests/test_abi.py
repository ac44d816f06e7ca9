"""C-ABI boundary checks that need no GPU: libcao.so builds, loads, exports every symbol include/cao.h
declares, and its host-side argument validation / call-order errors work."""
import ctypes as C
import os
import re
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2606_28372_b200 import build
    build.build()
    from paper_2606_28372_b200 import api
    return api.lib()


def _declared():
    src = open(os.path.join(ROOT, "include", "cao.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cao_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    from paper_2606_28372_b200 import api
    names = _declared()
    assert len(names) >= 28
    for nm in names:
        assert hasattr(L, nm), f"libcao.so does not export {nm}"
        assert nm in api.SIGNATURES, f"binding has no signature for {nm}"
    assert sorted(api.SIGNATURES) == names


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "cao.h"\nint main(void) { cao_hparams h; (void)h; return CAO_OK; }\n')
    import subprocess
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src),
                           "-o", str(tmp_path / "t.o")])


def test_host_side_validation(L):
    from paper_2606_28372_b200 import api
    h = C.c_void_p()
    assert L.cao_space_create(C.byref(h)) == 0
    vals = np.arange(300, dtype=np.int64)
    p = vals.ctypes.data_as(C.POINTER(C.c_int64))
    assert L.cao_space_add_param(h, b"a", p, 0) == -1                    # CAO_E_INVALID_ARG
    assert L.cao_space_add_param(h, b"a", p, 300) == -3                  # CAO_E_TOO_LARGE
    assert L.cao_space_add_param(h, b"a", p, 4) == 0
    bad = np.array([3], dtype=np.int32)                                  # ADD on an empty stack
    assert L.cao_space_add_constraint(h, bad.ctypes.data_as(api.pi32), 1) == -1
    assert b"malformed" in L.cao_last_error()
    oob = np.array([1, 7], dtype=np.int32)                               # PUSH_PARAM 7 with one parameter
    assert L.cao_space_add_constraint(h, oob.ctypes.data_as(api.pi32), 2) == -1
    ok = np.array([1, 0, 2, 2, 0, 14], dtype=np.int32)                   # p0 >= 2
    assert L.cao_space_add_constraint(h, ok.ctypes.data_as(api.pi32), 6) == 0
    tb = C.c_uint64()
    assert L.cao_space_table_bytes(h, C.byref(tb)) == -2                 # CAO_E_STATE: count first
    assert L.cao_space_build_fill(h, None, None) == -2
    bb, sb = C.c_uint64(), C.c_uint64()
    assert L.cao_space_build_workspace_bytes(h, C.byref(bb), C.byref(sb)) == 0
    assert bb.value >= 8 and bb.value % 256 == 0 and sb.value % 256 == 0
    V = C.c_uint64()
    assert L.cao_space_build_count(h, None, None, None, C.byref(V)) == -6    # CAO_E_WORKSPACE
    assert L.cao_space_add_param(h, b"b", p, 2) == -2                    # planned: no more params
    wb = C.c_uint64()
    assert L.cao_runs_workspace_bytes(h, 0, 8, 4, 10, C.byref(wb)) == -2  # space not built
    L.cao_space_destroy(h)


def test_too_large_space(L):
    h = C.c_void_p()
    assert L.cao_space_create(C.byref(h)) == 0
    vals = np.arange(256, dtype=np.int64)
    p = vals.ctypes.data_as(C.POINTER(C.c_int64))
    for _ in range(5):
        assert L.cao_space_add_param(h, b"x", p, 256) == 0               # 2^40 configs
    bb, sb = C.c_uint64(), C.c_uint64()
    assert L.cao_space_build_workspace_bytes(h, C.byref(bb), C.byref(sb)) == -3
    L.cao_space_destroy(h)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_28372_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "cao_oracle" not in txt, fn


def test_profile_class_names(L):
    """Every kernel class of cao_profile_read has a name that says which kernels it times; "" ends the list."""
    names = []
    while True:
        nm = L.cao_profile_name(len(names)).decode()
        if not nm:
            break
        names.append(nm)
    assert len(names) == 14 and len(set(names)) == 14
    assert "k_masks" in names[12] and "k_res_prefix" in names[13] and names[9] == "k_probe23"
    assert L.cao_profile_name(-1) == b""
