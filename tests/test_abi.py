"""CPU-side checks of the boundary: the library builds for sm_100a, loads without a GPU, exports
every symbol include/svf.h declares, and rejects bad arguments on the host (no compute calls)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def svf_lib():
    from paper_2606_22327_b200 import build
    path = build.build()
    return C.CDLL(path)


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "svf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(svf_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = _declared_functions()
    for need in ("svf_keys", "svf_admit", "svf_simulate"):
        assert need in names


def test_library_exports_every_declared_symbol(svf_lib):
    for name in _declared_functions():
        assert hasattr(svf_lib, name), f"{name} is declared in include/svf.h but not exported"


def test_binding_lists_the_same_exports(svf_lib):
    from paper_2606_22327_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_functions()


def test_status_strings_and_version(svf_lib):
    svf_lib.svf_status_string.restype = C.c_char_p
    svf_lib.svf_version.restype = C.c_char_p
    assert svf_lib.svf_status_string(0) == b"ok"
    for code in (1, 2, 3, 16, 17, 18, 19):
        assert len(svf_lib.svf_status_string(code)) > 0
    assert b"sm_100a" in svf_lib.svf_version()


def test_host_side_argument_errors_need_no_gpu(svf_lib):
    L = svf_lib
    L.svf_keys.restype = C.c_int
    L.svf_keys.argtypes = [C.c_int, C.c_int64] + [C.c_void_p] * 4 + [C.c_int32, C.c_int32] + [C.c_void_p] * 3
    assert L.svf_keys(7, 0, None, None, None, None, 1, 1, None, None, None) == 1       # unknown policy
    assert L.svf_keys(0, -1, None, None, None, None, 1, 1, None, None, None) == 1      # negative n
    assert L.svf_keys(1, 0, None, None, None, None, 0, 1, None, None, None) == 1       # 1-bit with O0 < 1
    assert L.svf_keys(1, 5, None, None, None, None, 1, 1, None, None, None) == 1       # 1-bit without bit
    assert L.svf_keys(0, 5, None, None, None, None, 1, 1, None, None, None) == 1       # null arrays
    L.svf_sort_workspace_bytes.restype = C.c_size_t
    L.svf_sort_workspace_bytes.argtypes = [C.c_int64, C.c_int, C.c_int]
    assert L.svf_sort_workspace_bytes(1000, 0, 64) > 8000
    assert L.svf_sort_workspace_bytes(1000, 8, 8) == 0
    L.svf_admit_workspace_bytes.restype = C.c_size_t
    L.svf_admit_workspace_bytes.argtypes = [C.c_int64, C.c_int64]
    assert L.svf_admit_workspace_bytes(1000, 100) > 16 * 1000
    assert L.svf_admit_workspace_bytes(-1, 0) == 0


def test_simulate_rejects_bad_host_arguments(svf_lib):
    from paper_2606_22327_b200.binding import _Result, _Trace
    L = svf_lib
    L.svf_simulate.restype = C.c_int
    L.svf_simulate.argtypes = [C.POINTER(_Trace), C.c_int, C.c_int64, C.POINTER(_Result), C.c_void_p,
                               C.c_size_t, C.c_void_p]
    tr = _Trace(1, 4, 4, None, None, None, None, None, 1, 1, None)
    res = _Result()
    assert L.svf_simulate(None, 0, 10, C.byref(res), None, 0, None) == 1
    assert L.svf_simulate(C.byref(tr), 9, 10, C.byref(res), None, 0, None) == 1           # policy
    assert L.svf_simulate(C.byref(tr), 0, -1, C.byref(res), None, 0, None) == 1           # M < 0
    assert L.svf_simulate(C.byref(tr), 1, 10, C.byref(res), None, 0, None) == 1           # 1-bit, no bit
    assert L.svf_simulate(C.byref(tr), 0, 10, C.byref(res), None, 0, None) == 1           # null offsets
    L.svf_simulate_workspace_bytes.restype = C.c_size_t
    L.svf_simulate_workspace_bytes.argtypes = [C.POINTER(_Trace)]
    assert L.svf_simulate_workspace_bytes(C.byref(tr)) > 0
    # several policies in one call
    L.svf_simulate_policies.restype = C.c_int
    L.svf_simulate_policies.argtypes = [C.POINTER(_Trace), C.c_int, C.POINTER(C.c_int), C.c_int64,
                                        C.POINTER(_Result), C.c_void_p, C.c_size_t, C.c_void_p]
    L.svf_simulate_policies_workspace_bytes.restype = C.c_size_t
    L.svf_simulate_policies_workspace_bytes.argtypes = [C.POINTER(_Trace), C.c_int]
    pol = (C.c_int * 2)(0, 3)
    outs = (_Result * 2)()
    assert L.svf_simulate_policies(C.byref(tr), 0, pol, 10, outs, None, 0, None) == 1     # n_policies < 1
    assert L.svf_simulate_policies(C.byref(tr), 9, pol, 10, outs, None, 0, None) == 1     # n_policies > 8
    assert L.svf_simulate_policies(C.byref(tr), 2, None, 10, outs, None, 0, None) == 1    # null policies
    bad = (C.c_int * 2)(0, 7)
    assert L.svf_simulate_policies(C.byref(tr), 2, bad, 10, outs, None, 0, None) == 1     # unknown policy
    assert L.svf_simulate_policies(C.byref(tr), 2, pol, 10, outs, None, 0, None) == 1     # null offsets
    w1 = L.svf_simulate_policies_workspace_bytes(C.byref(tr), 1)
    w4 = L.svf_simulate_policies_workspace_bytes(C.byref(tr), 4)
    assert w1 == L.svf_simulate_workspace_bytes(C.byref(tr)) and w4 > w1
    assert L.svf_simulate_policies_workspace_bytes(C.byref(tr), 0) == 0


def test_binding_refuses_cpu_tensors(svf_lib):
    import torch
    from paper_2606_22327_b200 import binding
    s = torch.ones(4, dtype=torch.int32)
    with pytest.raises(TypeError):
        binding.svf_keys(binding.SVF, s, s)
