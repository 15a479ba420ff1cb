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


# ---------------------------------------------------------------------------------------------
# workspace errors are found on the host, before the device is touched (include/svf.h conventions)
# ---------------------------------------------------------------------------------------------
def _sim_protos(L):
    from paper_2606_22327_b200.binding import _Result, _Trace
    L.svf_simulate.restype = C.c_int
    L.svf_simulate.argtypes = [C.POINTER(_Trace), C.c_int, C.c_int64, C.POINTER(_Result), C.c_void_p, C.c_size_t, C.c_void_p]
    L.svf_simulate_workspace_bytes.restype = C.c_size_t
    L.svf_simulate_workspace_bytes.argtypes = [C.POINTER(_Trace)]
    L.svf_volume_lower_bound.restype = C.c_int
    L.svf_volume_lower_bound.argtypes = [C.POINTER(_Trace), C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
    L.svf_volume_lower_bound_workspace_bytes.restype = C.c_size_t
    L.svf_volume_lower_bound_workspace_bytes.argtypes = [C.POINTER(_Trace)]
    L.svf_admit.restype = C.c_int
    L.svf_admit.argtypes = [C.c_int, C.c_int64, C.c_int32, C.c_int64] + [C.c_void_p] * 4 + [C.c_int32, C.c_int32, C.c_int64] + \
                           [C.c_void_p] * 7 + [C.c_size_t, C.c_void_p]
    L.svf_admit_workspace_bytes.restype = C.c_size_t
    L.svf_admit_workspace_bytes.argtypes = [C.c_int64, C.c_int64]
    L.svf_sort_words.restype = C.c_int
    L.svf_sort_words.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
    L.svf_sort_workspace_bytes.restype = C.c_size_t
    L.svf_sort_workspace_bytes.argtypes = [C.c_int64, C.c_int, C.c_int]
    return _Trace, _Result


# stand-ins for device pointers: the calls below must fail on the host before reading any of them
P0, P1, WS = 0x10000, 0x20000, 0x7000100


def test_short_and_unaligned_workspace_is_eworkspace(svf_lib):
    """SVF_EWORKSPACE from every call that takes `ws`: NULL, one byte short, and an UNALIGNED `ws`
    whose ws_bytes is smaller than the alignment pad (the size check must not wrap around)."""
    L = svf_lib
    _Trace, _Result = _sim_protos(L)
    EWS = 2
    tr = _Trace(3, 300, 100, P0, P0, P0, P0, P0, 1, 1, None)
    res = _Result()
    need = L.svf_simulate_workspace_bytes(C.byref(tr))
    assert need > 300 * 8
    for ws, nbytes in ((None, need), (WS, need - 257), (WS, 0), (WS + 1, 3), (WS + 1, 254), (WS + 255, need - 300)):
        assert L.svf_simulate(C.byref(tr), 0, 1000, C.byref(res), ws, nbytes, None) == EWS, (ws, nbytes)
        assert L.svf_volume_lower_bound(C.byref(tr), P1, None, ws, nbytes, None) == EWS, (ws, nbytes)
    need = L.svf_admit_workspace_bytes(500, 40)
    for ws, nbytes in ((None, need), (WS, need - 257), (WS + 1, 3), (WS + 8, 200)):
        rc = L.svf_admit(0, 1000, 0, 500, P0, P0, P0, None, 1, 1, 40, P0, P0, P1, None, None, None, ws, nbytes, None)
        assert rc == EWS, (ws, nbytes)
    need = L.svf_sort_workspace_bytes(5000, 0, 64)
    for ws, nbytes in ((None, need), (WS, need - 257), (WS + 1, 3), (WS + 8, 200)):
        assert L.svf_sort_words(5000, P0, P1, 0, 64, ws, nbytes, None) == EWS, (ws, nbytes)


def test_onebit_without_requests_needs_no_bit_array(svf_lib):
    """n = 0 under SVF_SVF_1BIT with bit = NULL is NOT an argument error (svf.h conventions; the oracle
    takes the same call, tests/test_oracle_pins.py); O0, O1 >= 1 are still required."""
    L = svf_lib
    _Trace, _Result = _sim_protos(L)
    L.svf_keys.restype = C.c_int
    L.svf_keys.argtypes = [C.c_int, C.c_int64] + [C.c_void_p] * 4 + [C.c_int32, C.c_int32] + [C.c_void_p] * 3
    assert L.svf_keys(1, 0, None, None, None, None, 2, 8, None, None, None) != 1
    assert L.svf_keys(1, 0, None, None, None, None, 0, 8, None, None, None) == 1
    rc = L.svf_admit(1, 1000, 0, 0, None, None, None, None, 2, 8, 0, None, None, P1, None, None, None, WS, 1 << 20, None)
    assert rc != 1
    tr = _Trace(2, 0, 0, P0, None, None, None, None, 2, 8, None)
    assert L.svf_simulate(C.byref(tr), 1, 1000, C.byref(_Result()), WS, 1 << 20, None) != 1


_NO_DEVICE_SCRIPT = r"""
import ctypes as C, sys
sys.path.insert(0, {root!r})
from paper_2606_22327_b200.binding import _Result, _Trace
L = C.CDLL({lib!r})
P0, P1, WS, BIG = 0x10000, 0x20000, 0x7000100, 1 << 30
L.svf_keys.restype = C.c_int
L.svf_keys.argtypes = [C.c_int, C.c_int64] + [C.c_void_p] * 4 + [C.c_int32, C.c_int32] + [C.c_void_p] * 3
L.svf_simulate.restype = C.c_int
L.svf_simulate.argtypes = [C.POINTER(_Trace), C.c_int, C.c_int64, C.POINTER(_Result), C.c_void_p, C.c_size_t, C.c_void_p]
L.svf_simulate_policies.restype = C.c_int
L.svf_simulate_policies.argtypes = [C.POINTER(_Trace), C.c_int, C.POINTER(C.c_int), C.c_int64, C.POINTER(_Result), C.c_void_p, C.c_size_t, C.c_void_p]
L.svf_volume_lower_bound.restype = C.c_int
L.svf_volume_lower_bound.argtypes = [C.POINTER(_Trace), C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
L.svf_admit.restype = C.c_int
L.svf_admit.argtypes = [C.c_int, C.c_int64, C.c_int32, C.c_int64] + [C.c_void_p] * 4 + [C.c_int32, C.c_int32, C.c_int64] + [C.c_void_p] * 7 + [C.c_size_t, C.c_void_p]
L.svf_sort_words.restype = C.c_int
L.svf_sort_words.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
tr = _Trace(3, 300, 100, P0, P0, P0, P0, P0, 1, 1, None)
res = _Result()
pol = (C.c_int * 2)(0, 3)
outs = (_Result * 2)()
rcs = [L.svf_keys(0, 100, P0, P0, None, None, 1, 1, P1, None, None),
       L.svf_simulate(C.byref(tr), 0, 1000, C.byref(res), WS, BIG, None),
       L.svf_simulate(C.byref(tr), 0, 1 << 31, C.byref(res), WS, BIG, None),
       L.svf_simulate_policies(C.byref(tr), 2, pol, 1000, outs, WS, BIG, None),
       L.svf_volume_lower_bound(C.byref(tr), P1, None, WS, BIG, None),
       L.svf_admit(0, 1000, 0, 500, P0, P0, P0, None, 1, 1, 40, P0, P0, P1, None, None, None, WS, BIG, None),
       L.svf_sort_words(5000, P0, P1, 0, 64, WS, BIG, None)]
print(",".join(str(r) for r in rcs))
"""


def test_compute_calls_return_ecuda_without_a_device(svf_lib):
    """No CPU fallback: with no CUDA device visible every compute entry point returns SVF_ECUDA (3)
    and touches none of its buffers.  Run in a child process with CUDA_VISIBLE_DEVICES empty, so the
    test says the same on the GPU box."""
    import subprocess
    import sys
    from paper_2606_22327_b200 import build
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    out = subprocess.run([sys.executable, "-c", _NO_DEVICE_SCRIPT.format(root=ROOT, lib=build.LIB)], env=env,
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    assert out.stdout.strip() == ",".join(["3"] * 7), out.stdout


def test_static_admit_checks_arguments_and_its_size_limit_on_the_host(svf_lib):
    """svf_admit_static (scratch inside the library, for callers that may not allocate): argument
    errors and the stated maximum are found before the device is touched; the maximum fits the array."""
    L = svf_lib
    f = L.svf_admit_static
    f.restype = C.c_int
    f.argtypes = [C.c_int, C.c_int64, C.c_int32, C.c_int64] + [C.c_void_p] * 4 + [C.c_int32, C.c_int32, C.c_int64] + [C.c_void_p] * 7
    k = C.c_int64(0)
    kp = C.addressof(k)
    args = lambda policy, n_wait, n_run, out=kp: (policy, 100, 0, n_wait, None, None, None, None, 1, 1, n_run, None, None, out, None, None, None, None)
    assert f(*args(9, 0, 0)) == 1                      # unknown policy
    assert f(*args(0, -1, 0)) == 1                     # negative size
    assert f(*args(0, 0, 0, None)) == 1                # nowhere to write the answer
    assert f(*args(0, 5, 0)) == 1                      # null arrays
    buf = (C.c_int32 * 70000)()
    p = C.addressof(buf)
    wide = lambda n_wait, n_run: (0, 100, 0, n_wait, p, p, p, None, 1, 1, n_run, p, p, kp, None, None, None, None)
    assert f(*wide(65537, 0)) == 2                     # beyond SVF_ADMIT_STATIC_MAX_WAIT
    assert f(*wide(10, 8193)) == 2                     # beyond SVF_ADMIT_STATIC_MAX_RUN
    hdr = open(os.path.join(ROOT, "include", "svf.h")).read()
    mw = int(re.search(r"SVF_ADMIT_STATIC_MAX_WAIT\s+(\d+)", hdr).group(1))
    mr = int(re.search(r"SVF_ADMIT_STATIC_MAX_RUN\s+(\d+)", hdr).group(1))
    sh = int(re.search(r"SVF_ADMIT_STATIC_BYTES\s+\((\d+) << 20\)", hdr).group(1))
    L.svf_admit_workspace_bytes.restype = C.c_size_t
    L.svf_admit_workspace_bytes.argtypes = [C.c_int64, C.c_int64]
    assert (mw, mr) == (65536, 8192)
    assert L.svf_admit_workspace_bytes(mw, mr) <= sh << 20


def test_simulate_workspace_covers_the_layout_of_every_budget(svf_lib):
    """svf_simulate*_workspace_bytes is taken without knowing M, yet M picks the kernel form and the forms
    carve different scratch.  Sweep M (around every breakpoint of the group-width rule, 512 tokens per
    estimated running request, and across 2^30), instance sizes around every state-placement limit,
    instance counts from one to many waves and 1 / 4 / 8 policies: no budget may need more than the
    size the caller was told to provide."""
    from paper_2606_22327_b200 import binding
    L = svf_lib
    L.svf_simulate_policies_workspace_bytes.restype = C.c_size_t
    L.svf_simulate_policies_workspace_bytes.argtypes = [C.POINTER(binding._Trace), C.c_int]
    L.svf_simulate_layout_bytes.restype = C.c_size_t
    L.svf_simulate_layout_bytes.argtypes = [C.POINTER(binding._Trace), C.c_int, C.c_int64]
    budgets = [0, 1, 511, 512, 2 ** 30 - 1, 2 ** 30, 2 ** 30 + 1, 2 ** 40]
    for r in (511, 512, 513, 767, 768, 769, 1023, 1024, 1025, 1599, 1600, 1601, 2047, 2048, 2049, 4096, 8192, 8193, 100_000):
        budgets += [512 * r - 1, 512 * r, 512 * r + 511, 512 * (r + 1)]
    checked = 0
    for mx in (1, 31, 33, 500, 1000, 1024, 1025, 2048, 2049, 4096, 4097, 8192, 8193, 20_000, 200_000):
        for I in (1, 2, 7, 148, 1000, 4096, 100_000):
            N = min(I * mx, 2 ** 29)
            for P in (1, 4, 8):
                tr = binding._Trace()
                tr.n_instances, tr.n_requests, tr.max_instance = I, N, min(mx, N)
                cap = L.svf_simulate_policies_workspace_bytes(C.byref(tr), P)
                assert cap > 0
                for M in budgets:
                    need = L.svf_simulate_layout_bytes(C.byref(tr), P, M)
                    assert 0 < need <= cap, f"max_instance {mx}, I {I}, P {P}, M {M}: layout {need} > workspace {cap}"
                    checked += 1
    assert checked > 20_000
    assert L.svf_simulate_layout_bytes(None, 1, 0) == 0 and L.svf_simulate_layout_bytes(C.byref(tr), 9, 0) == 0
