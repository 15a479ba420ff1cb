"""ctypes wrapper around the CPU ORACLE ``oracle/svf_ref.c`` (test infrastructure only).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this module.  It never imports the CUDA binding; the two share no code.

``build()`` compiles ``svf_ref.c`` with gcc into ``oracle/libsvf_ref.so`` (building the checker
is not using it: ``__graft_entry__.build()`` calls this too).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "svf_ref.c")
_LIB = os.path.join(_DIR, "libsvf_ref.so")

SVF, SVF_1BIT, SJF, FCFS = 0, 1, 2, 3
POLICY_NAMES = {SVF: "svf", SVF_1BIT: "svf_1bit", SJF: "sjf", FCFS: "fcfs"}
OK, EINVAL, ERANGE, EUNSORTED, EINFEASIBLE, EOVERFLOW = 0, 1, 16, 17, 18, 19

FEAS_LITERAL, FEAS_COMPLETION = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP for instance-parallel batches)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.svf_ref_max_threads.restype = C.c_int
    return _lib


def _p(arr, ctype):
    return None if arr is None else arr.ctypes.data_as(C.POINTER(ctype))


def _i32(x):
    return None if x is None else np.ascontiguousarray(x, dtype=np.int32)


def _u8(x):
    return None if x is None else np.ascontiguousarray(x, dtype=np.uint8)


def max_threads() -> int:
    return int(lib().svf_ref_max_threads())


def keys(policy, s, o, a=None, bit=None, O0=1, O1=1):
    """Packed words ``(key << 32) + id`` (Eq. 1 / Eq. 2 / SJF / FCFS keys).  Returns (rc, words)."""
    s, o, a, bit = _i32(s), _i32(o), _i32(a), _u8(bit)
    n = len(s)
    words = np.zeros(n, dtype=np.uint64)
    rc = lib().svf_ref_keys(C.c_int(policy), C.c_int64(n), _p(s, C.c_int32), _p(o, C.c_int32),
                            _p(a, C.c_int32), _p(bit, C.c_uint8), C.c_int32(O0), C.c_int32(O1),
                            _p(words, C.c_uint64))
    return rc, words


def feasible(kv, rem, M, mode=FEAS_COMPLETION) -> bool:
    kv = np.ascontiguousarray(kv, dtype=np.int64)
    rem = np.ascontiguousarray(rem, dtype=np.int64)
    return bool(lib().svf_ref_feasible(C.c_int(mode), C.c_int64(len(kv)), _p(kv, C.c_int64),
                                       _p(rem, C.c_int64), C.c_int64(M)))


def admit(policy, M, t, w_s, w_o, w_a, w_bit, O0, O1, r_kv, r_rem, mode=FEAS_COMPLETION):
    """One stateless admission decision.  Returns (rc, admitted_idx[int32], sorted_words)."""
    w_s, w_o, w_a, w_bit = _i32(w_s), _i32(w_o), _i32(w_a), _u8(w_bit)
    r_kv, r_rem = _i32(r_kv), _i32(r_rem)
    nw, nr = len(w_s), len(r_kv)
    n_adm = C.c_int64(0)
    idx = np.full(max(nw, 1), -1, dtype=np.int32)
    words = np.zeros(max(nw, 1), dtype=np.uint64)
    rc = lib().svf_ref_admit(C.c_int(policy), C.c_int64(M), C.c_int32(t), C.c_int(mode),
                             C.c_int64(nw), _p(w_s, C.c_int32), _p(w_o, C.c_int32),
                             _p(w_a, C.c_int32), _p(w_bit, C.c_uint8), C.c_int32(O0),
                             C.c_int32(O1), C.c_int64(nr), _p(r_kv, C.c_int32),
                             _p(r_rem, C.c_int32), C.byref(n_adm), _p(idx, C.c_int32),
                             _p(words, C.c_uint64))
    return rc, idx[: n_adm.value].copy(), words[:nw].copy()


@dataclass
class SimResult:
    start: np.ndarray
    finish: np.ndarray
    total_latency: np.ndarray
    p99_latency: np.ndarray
    makespan: np.ndarray
    peak_kv: np.ndarray
    rounds: np.ndarray
    decisions: np.ndarray
    status: np.ndarray


def simulate(trace, policy, M=None, mode=FEAS_COMPLETION, n_threads=1, output_key="trace") -> SimResult:
    """Run the time-stepped simulator on every instance of ``trace`` (a traces.Trace).
    ``output_key``: predicted output lengths used for the SVF / SJF key only (default: the
    trace's own ``output_key`` if it has one; None = the true lengths)."""
    if isinstance(output_key, str):
        output_key = getattr(trace, "output_key", None)
    ok = _i32(output_key)
    M = trace.M if M is None else M
    I, N = trace.n_instances, trace.n_requests
    off = np.ascontiguousarray(trace.offsets, dtype=np.int64)
    a, s, o, b = _i32(trace.arrival), _i32(trace.prompt), _i32(trace.output), _u8(trace.bit)
    r = SimResult(np.full(N, -1, np.int32), np.full(N, -1, np.int32), np.zeros(I, np.int64),
                  np.zeros(I, np.int64), np.zeros(I, np.int32), np.zeros(I, np.int64),
                  np.zeros(I, np.int64), np.zeros(I, np.int64), np.zeros(I, np.int32))
    rc = lib().svf_ref_simulate_pred(
        C.c_int64(I), _p(off, C.c_int64), _p(a, C.c_int32), _p(s, C.c_int32), _p(o, C.c_int32),
        _p(ok, C.c_int32), _p(b, C.c_uint8), C.c_int32(trace.O0), C.c_int32(trace.O1), C.c_int(policy),
        C.c_int64(M), C.c_int(mode), C.c_int(n_threads),
        _p(r.start, C.c_int32), _p(r.finish, C.c_int32), _p(r.total_latency, C.c_int64),
        _p(r.p99_latency, C.c_int64), _p(r.makespan, C.c_int32), _p(r.peak_kv, C.c_int64),
        _p(r.rounds, C.c_int64), _p(r.decisions, C.c_int64), _p(r.status, C.c_int32))
    if rc != OK:
        raise RuntimeError(f"svf_ref_simulate failed: {rc}")
    return r


def bruteforce_opt(s, o, M):
    """Hindsight optimum TEL of a tiny burst instance (IP 3a-3d).  Returns (opt, start, nodes)."""
    s, o = _i32(s), _i32(o)
    n = len(s)
    opt, nodes = C.c_int64(0), C.c_int64(0)
    start = np.zeros(n, dtype=np.int32)
    rc = lib().svf_ref_bruteforce_opt(C.c_int64(n), _p(s, C.c_int32), _p(o, C.c_int32),
                                      C.c_int64(M), C.byref(opt), _p(start, C.c_int32),
                                      C.byref(nodes))
    if rc != OK:
        raise RuntimeError(f"svf_ref_bruteforce_opt failed: {rc}")
    return int(opt.value), start, int(nodes.value)


def volume_lower_bound(trace):
    """Prop. 3.1 (Eq. 5): LB_j = sum_j sum_{i<=j} vol_(i) per instance, so that for burst input
    M * TEL(any schedule) >= LB.  Returns (lb[int64 I], status[int32 I])."""
    I = trace.n_instances
    off = np.ascontiguousarray(trace.offsets, dtype=np.int64)
    s, o = _i32(trace.prompt), _i32(trace.output)
    lb = np.zeros(I, np.int64)
    st = np.zeros(I, np.int32)
    rc = lib().svf_ref_volume_lower_bound(C.c_int64(I), _p(off, C.c_int64), _p(s, C.c_int32), _p(o, C.c_int32),
                                          _p(lb, C.c_int64), _p(st, C.c_int32))
    if rc != OK:
        raise RuntimeError(f"svf_ref_volume_lower_bound failed: {rc}")
    return lb, st
