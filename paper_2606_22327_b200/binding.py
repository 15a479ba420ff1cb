"""Thin ctypes binding over ``csrc/libsvf_b200.so`` (the C ABI of ``include/svf.h``).

Argument marshalling only: every step of the hot path runs in the CUDA kernels.  PyTorch supplies
device memory and streams.  There is no CPU fallback: a missing library, a CPU tensor or a box
without a CUDA device raises.  Function names mirror the C entry points.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import torch

_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_DIR, "csrc", "libsvf_b200.so")

SVF, SVF_1BIT, SJF, FCFS = 0, 1, 2, 3
POLICY_NAMES = {SVF: "svf", SVF_1BIT: "svf_1bit", SJF: "sjf", FCFS: "fcfs"}
OK, EINVAL, EWORKSPACE, ECUDA = 0, 1, 2, 3
ERANGE, EUNSORTED, EINFEASIBLE, EOVERFLOW = 16, 17, 18, 19

EXPORTS = ("svf_keys", "svf_admit_workspace_bytes", "svf_admit", "svf_admit_static", "svf_simulate_workspace_bytes",
           "svf_simulate", "svf_simulate_policies_workspace_bytes", "svf_simulate_policies", "svf_simulate_layout_bytes",
           "svf_volume_lower_bound_workspace_bytes", "svf_volume_lower_bound", "svf_sort_workspace_bytes", "svf_sort_words", "svf_last_launch_count",
           "svf_status_string", "svf_version", "svf_set_profiling", "svf_simulate_phase_ms",
           "svf_simulate_work_counts", "svf_admit_phase_ms")


class SvfError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {status_string(code)} ({code})")


class _Trace(C.Structure):
    _fields_ = [("n_instances", C.c_int64), ("n_requests", C.c_int64), ("max_instance", C.c_int64),
                ("offsets", C.c_void_p), ("arrival", C.c_void_p), ("prompt", C.c_void_p),
                ("output", C.c_void_p), ("bit", C.c_void_p), ("O0", C.c_int32), ("O1", C.c_int32),
                ("output_key", C.c_void_p)]


class _Result(C.Structure):
    _fields_ = [("start", C.c_void_p), ("finish", C.c_void_p), ("total_latency", C.c_void_p),
                ("p99_latency", C.c_void_p), ("makespan", C.c_void_p), ("peak_kv", C.c_void_p),
                ("rounds", C.c_void_p), ("decisions", C.c_void_p), ("status", C.c_void_p)]


_lib = None


def lib():
    """Load the shared library (raises if it has not been built: there is no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with "
                               "`python -m paper_2606_22327_b200.build` (no CPU fallback exists)")
        L = C.CDLL(LIB_PATH)
        L.svf_keys.restype = C.c_int
        L.svf_keys.argtypes = [C.c_int, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                               C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.svf_admit_workspace_bytes.restype = C.c_size_t
        L.svf_admit_workspace_bytes.argtypes = [C.c_int64, C.c_int64]
        L.svf_admit.restype = C.c_int
        L.svf_admit.argtypes = [C.c_int, C.c_int64, C.c_int32, C.c_int64, C.c_void_p, C.c_void_p,
                                C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_void_p,
                                C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                C.c_void_p, C.c_size_t, C.c_void_p]
        L.svf_admit_static.restype = C.c_int
        L.svf_admit_static.argtypes = [C.c_int, C.c_int64, C.c_int32, C.c_int64, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int64,
                                       C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p]
        L.svf_simulate_workspace_bytes.restype = C.c_size_t
        L.svf_simulate_workspace_bytes.argtypes = [C.POINTER(_Trace)]
        L.svf_simulate.restype = C.c_int
        L.svf_simulate.argtypes = [C.POINTER(_Trace), C.c_int, C.c_int64, C.POINTER(_Result),
                                   C.c_void_p, C.c_size_t, C.c_void_p]
        L.svf_simulate_policies_workspace_bytes.restype = C.c_size_t
        L.svf_simulate_policies_workspace_bytes.argtypes = [C.POINTER(_Trace), C.c_int]
        L.svf_simulate_policies.restype = C.c_int
        L.svf_simulate_policies.argtypes = [C.POINTER(_Trace), C.c_int, C.POINTER(C.c_int), C.c_int64,
                                            C.POINTER(_Result), C.c_void_p, C.c_size_t, C.c_void_p]
        L.svf_simulate_layout_bytes.restype = C.c_size_t
        L.svf_simulate_layout_bytes.argtypes = [C.POINTER(_Trace), C.c_int, C.c_int64]
        L.svf_volume_lower_bound_workspace_bytes.restype = C.c_size_t
        L.svf_volume_lower_bound_workspace_bytes.argtypes = [C.POINTER(_Trace)]
        L.svf_volume_lower_bound.restype = C.c_int
        L.svf_volume_lower_bound.argtypes = [C.POINTER(_Trace), C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t,
                                             C.c_void_p]
        L.svf_sort_workspace_bytes.restype = C.c_size_t
        L.svf_sort_workspace_bytes.argtypes = [C.c_int64, C.c_int, C.c_int]
        L.svf_sort_words.restype = C.c_int
        L.svf_sort_words.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                     C.c_void_p, C.c_size_t, C.c_void_p]
        L.svf_last_launch_count.restype = C.c_int64
        L.svf_last_launch_count.argtypes = [C.c_int]
        L.svf_status_string.restype = C.c_char_p
        L.svf_status_string.argtypes = [C.c_int]
        L.svf_version.restype = C.c_char_p
        L.svf_set_profiling.restype = None
        L.svf_set_profiling.argtypes = [C.c_int]
        L.svf_simulate_phase_ms.restype = C.c_int
        L.svf_simulate_phase_ms.argtypes = [C.POINTER(C.c_float)]
        L.svf_simulate_work_counts.restype = C.c_int
        L.svf_simulate_work_counts.argtypes = [C.POINTER(C.c_uint64)]
        L.svf_admit_phase_ms.restype = C.c_int
        L.svf_admit_phase_ms.argtypes = [C.POINTER(C.c_float)]
        _lib = L
    return _lib


def status_string(code: int) -> str:
    return lib().svf_status_string(int(code)).decode()


def version() -> str:
    return lib().svf_version().decode()


def set_profiling(mode) -> None:
    """0/False off, 1/True phase events, 2 phase events + algorithmic work counts."""
    lib().svf_set_profiling(int(mode))


def simulate_work_counts():
    """(E, U, evaluations, blocked) of the last svf_simulate call made under set_profiling(2): running
    entries examined over all head evaluations, running entries updated over all admissions, head
    evaluations performed, and how many of them found the head blocked."""
    buf = (C.c_uint64 * 4)()
    _check(lib().svf_simulate_work_counts(buf), "svf_simulate_work_counts")
    return tuple(int(x) for x in buf)


def simulate_phase_ms():
    """(phase A, phase B, phase C, whole call) in ms for the last profiled svf_simulate call."""
    buf = (C.c_float * 4)()
    _check(lib().svf_simulate_phase_ms(buf), "svf_simulate_phase_ms")
    return tuple(float(x) for x in buf)


def admit_phase_ms():
    """(keys + validation, sorts, admission, whole call) in ms for the last profiled svf_admit call."""
    buf = (C.c_float * 4)()
    _check(lib().svf_admit_phase_ms(buf), "svf_admit_phase_ms")
    return tuple(float(x) for x in buf)


def last_launch_count(which: int) -> int:
    return int(lib().svf_last_launch_count(which))


def _ptr(t: Optional[torch.Tensor], dtype, name: str):
    if t is None:
        return None
    if not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor (the library has no CPU path)")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _hold(ws: torch.Tensor, stream) -> None:
    """A workspace allocated inside a call is dropped when the call returns while its kernels are only
    enqueued: tell the caching allocator which stream still uses it (same-stream reuse is ordered)."""
    if stream is not None and stream != torch.cuda.current_stream(ws.device):
        ws.record_stream(stream)


def _check(rc: int, where: str):
    if rc != OK:
        raise SvfError(rc, where)


# ---------------------------------------------------------------------------------------------
# svf_keys
# ---------------------------------------------------------------------------------------------
def svf_keys(policy, s, o, a=None, bit=None, O0=1, O1=1, words_out=None, status_out=None, stream=None):
    """words[i] = (key_i << 32) + i on the device.  Returns (words, status[1])."""
    ref = s if s is not None else (o if o is not None else a)
    n = int(ref.numel())
    dev = ref.device
    if words_out is None:
        words_out = torch.empty(n, dtype=torch.int64, device=dev)
    if status_out is None:
        status_out = torch.empty(1, dtype=torch.int32, device=dev)
    rc = lib().svf_keys(int(policy), n, _ptr(s, torch.int32, "s"), _ptr(o, torch.int32, "o"),
                        _ptr(a, torch.int32, "a"), _ptr(bit, torch.uint8, "bit"), int(O0), int(O1),
                        _ptr(words_out, torch.int64, "words_out"),
                        _ptr(status_out, torch.int32, "status_out"), _stream(stream))
    _check(rc, "svf_keys")
    return words_out, status_out


# ---------------------------------------------------------------------------------------------
# svf_sort_words
# ---------------------------------------------------------------------------------------------
def svf_sort_words(words, bit_lo=0, bit_hi=64, out=None, ws=None, stream=None):
    n = int(words.numel())
    if out is None:
        out = torch.empty_like(words)
    need = int(lib().svf_sort_workspace_bytes(n, int(bit_lo), int(bit_hi)))
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 256), dtype=torch.uint8, device=words.device)
    rc = lib().svf_sort_words(n, _ptr(words, torch.int64, "words"), _ptr(out, torch.int64, "out"),
                              int(bit_lo), int(bit_hi), C.c_void_p(ws.data_ptr()), ws.numel(),
                              _stream(stream))
    _check(rc, "svf_sort_words")
    _hold(ws, stream)
    return out


# ---------------------------------------------------------------------------------------------
# svf_admit
# ---------------------------------------------------------------------------------------------
@dataclass
class AdmitOut:
    n_admitted: torch.Tensor      # int64 [1]
    admitted_idx: torch.Tensor    # int32 [n_wait]
    sorted_words: Optional[torch.Tensor]
    status: torch.Tensor          # int32 [1]


def svf_admit_workspace_bytes(n_wait: int, n_run: int) -> int:
    return int(lib().svf_admit_workspace_bytes(int(n_wait), int(n_run)))


def svf_admit(policy, M, t, w_s, w_o, w_a, w_bit, O0, O1, r_kv, r_rem, want_sorted=True, ws=None,
              out: Optional[AdmitOut] = None, stream=None) -> AdmitOut:
    nw, nr = int(w_s.numel()), int(r_kv.numel())
    dev = w_s.device
    if out is None:
        out = AdmitOut(torch.zeros(1, dtype=torch.int64, device=dev),
                       torch.full((max(nw, 1),), -1, dtype=torch.int32, device=dev),
                       torch.zeros(max(nw, 1), dtype=torch.int64, device=dev) if want_sorted else None,
                       torch.zeros(1, dtype=torch.int32, device=dev))
    need = svf_admit_workspace_bytes(nw, nr)
    if ws is None or ws.numel() < need:
        ws = torch.empty(need, dtype=torch.uint8, device=dev)
    rc = lib().svf_admit(int(policy), int(M), int(t), nw, _ptr(w_s, torch.int32, "w_s"),
                         _ptr(w_o, torch.int32, "w_o"), _ptr(w_a, torch.int32, "w_a"),
                         _ptr(w_bit, torch.uint8, "w_bit"), int(O0), int(O1), nr,
                         _ptr(r_kv, torch.int32, "r_kv"), _ptr(r_rem, torch.int32, "r_rem"),
                         _ptr(out.n_admitted, torch.int64, "n_admitted"),
                         _ptr(out.admitted_idx, torch.int32, "admitted_idx"),
                         _ptr(out.sorted_words, torch.int64, "sorted_words"),
                         _ptr(out.status, torch.int32, "status"), C.c_void_p(ws.data_ptr()),
                         ws.numel(), _stream(stream))
    _check(rc, "svf_admit")
    _hold(ws, stream)
    out._ws = ws  # keep the scratch alive until the caller drops the result
    return out


ADMIT_STATIC_MAX_WAIT, ADMIT_STATIC_MAX_RUN = 65536, 8192     # the limits include/svf.h states


def svf_admit_static(policy, M, t, w_s, w_o, w_a, w_bit, O0, O1, r_kv, r_rem, out: AdmitOut,
                     stream=None) -> AdmitOut:
    """svf_admit for a caller that must not allocate device memory (a scheduler inside a serving
    engine whose KV-cache pool already owns the HBM, where cudaMalloc can fail and would stall the
    decode stream).  The scratch is a fixed array inside the library, so this binding allocates
    nothing either: `out` (an AdmitOut you made once at start-up; sorted_words may be None) is
    required and is filled in place.  Raises SvfError(EWORKSPACE) above 65,536 waiting or 8,192
    running requests.  Calls share the one array per GPU: keep them on one stream, or order them."""
    nw, nr = int(w_s.numel()), int(r_kv.numel())
    rc = lib().svf_admit_static(int(policy), int(M), int(t), nw, _ptr(w_s, torch.int32, "w_s"),
                                _ptr(w_o, torch.int32, "w_o"), _ptr(w_a, torch.int32, "w_a"),
                                _ptr(w_bit, torch.uint8, "w_bit"), int(O0), int(O1), nr,
                                _ptr(r_kv, torch.int32, "r_kv"), _ptr(r_rem, torch.int32, "r_rem"),
                                _ptr(out.n_admitted, torch.int64, "n_admitted"),
                                _ptr(out.admitted_idx, torch.int32, "admitted_idx"),
                                _ptr(out.sorted_words, torch.int64, "sorted_words"),
                                _ptr(out.status, torch.int32, "status"), _stream(stream))
    _check(rc, "svf_admit_static")
    return out


# ---------------------------------------------------------------------------------------------
# svf_simulate
# ---------------------------------------------------------------------------------------------
@dataclass
class DeviceTrace:
    """The svf_trace_t arrays on the device (torch owns the memory)."""
    offsets: torch.Tensor   # int64 [I+1]
    arrival: torch.Tensor   # int32 [N]
    prompt: torch.Tensor    # int32 [N]
    output: torch.Tensor    # int32 [N]
    bit: Optional[torch.Tensor]   # uint8 [N]
    n_instances: int
    n_requests: int
    max_instance: int
    O0: int
    O1: int
    M: int
    output_key: Optional[torch.Tensor] = None   # int32 [N] predicted lengths (SVF / SJF key only)

    @staticmethod
    def from_host(trace, device="cuda", pinned=None, non_blocking=False) -> "DeviceTrace":
        """Copy a ``traces.Trace`` (numpy) to the device.  ``pinned``: optional dict of pinned
        host tensors to copy from (the end-to-end leg of bench.py)."""
        def up(name, arr, dt):
            src = pinned[name] if pinned is not None else torch.from_numpy(arr)
            return src.to(device=device, dtype=dt, non_blocking=non_blocking)
        return DeviceTrace(up("offsets", trace.offsets, torch.int64), up("arrival", trace.arrival, torch.int32),
                           up("prompt", trace.prompt, torch.int32), up("output", trace.output, torch.int32),
                           up("bit", trace.bit, torch.uint8), trace.n_instances, trace.n_requests,
                           trace.max_n, int(trace.O0), int(trace.O1), int(trace.M),
                           None if getattr(trace, "output_key", None) is None
                           else torch.from_numpy(trace.output_key).to(device=device, dtype=torch.int32))

    def nbytes(self) -> int:
        return sum(int(t.numel() * t.element_size()) for t in
                   (self.offsets, self.arrival, self.prompt, self.output, self.bit) if t is not None)

    def c_struct(self) -> _Trace:
        return _Trace(self.n_instances, self.n_requests, self.max_instance,
                      self.offsets.data_ptr(), self.arrival.data_ptr(), self.prompt.data_ptr(),
                      self.output.data_ptr(), self.bit.data_ptr() if self.bit is not None else None,
                      self.O0, self.O1,
                      self.output_key.data_ptr() if self.output_key is not None else None)


RESULT_FIELDS = ("start", "finish", "total_latency", "p99_latency", "makespan", "peak_kv", "rounds",
                 "decisions", "status")
_PER_REQUEST = {"start": torch.int32, "finish": torch.int32}
_PER_INSTANCE = {"total_latency": torch.int64, "p99_latency": torch.int64, "makespan": torch.int32,
                 "peak_kv": torch.int64, "rounds": torch.int64, "decisions": torch.int64,
                 "status": torch.int32}


@dataclass
class SimOut:
    start: Optional[torch.Tensor] = None
    finish: Optional[torch.Tensor] = None
    total_latency: Optional[torch.Tensor] = None
    p99_latency: Optional[torch.Tensor] = None
    makespan: Optional[torch.Tensor] = None
    peak_kv: Optional[torch.Tensor] = None
    rounds: Optional[torch.Tensor] = None
    decisions: Optional[torch.Tensor] = None
    status: Optional[torch.Tensor] = None

    @staticmethod
    def alloc(dt: DeviceTrace, want=RESULT_FIELDS) -> "SimOut":
        dev = dt.offsets.device
        o = SimOut()
        for k in want:
            if k in _PER_REQUEST:
                setattr(o, k, torch.full((max(dt.n_requests, 1),), -7, dtype=_PER_REQUEST[k], device=dev))
            else:
                setattr(o, k, torch.full((max(dt.n_instances, 1),), -7, dtype=_PER_INSTANCE[k], device=dev))
        return o

    def c_struct(self) -> _Result:
        g = lambda k: (getattr(self, k).data_ptr() if getattr(self, k) is not None else None)
        return _Result(*[g(k) for k in RESULT_FIELDS])

    def nbytes(self) -> int:
        return sum(int(getattr(self, k).numel() * getattr(self, k).element_size())
                   for k in RESULT_FIELDS if getattr(self, k) is not None)


def svf_simulate_workspace_bytes(dt: DeviceTrace) -> int:
    tr = dt.c_struct()
    return int(lib().svf_simulate_workspace_bytes(C.byref(tr)))


def svf_simulate(dt: DeviceTrace, policy: int, M: Optional[int] = None, out: Optional[SimOut] = None,
                 ws: Optional[torch.Tensor] = None, want=RESULT_FIELDS, stream=None) -> SimOut:
    """Enqueue one batched simulation; results are valid after the stream synchronises."""
    if not dt.offsets.is_cuda:
        raise TypeError("svf_simulate needs device tensors (the library has no CPU path)")
    M = dt.M if M is None else int(M)
    if out is None:
        out = SimOut.alloc(dt, want)
    need = svf_simulate_workspace_bytes(dt)
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 256), dtype=torch.uint8, device=dt.offsets.device)
    tr, res = dt.c_struct(), out.c_struct()
    rc = lib().svf_simulate(C.byref(tr), int(policy), M, C.byref(res), C.c_void_p(ws.data_ptr()),
                            ws.numel(), _stream(stream))
    _check(rc, "svf_simulate")
    _hold(ws, stream)
    out._ws = ws  # keep the scratch alive until the caller drops the result
    return out


def svf_simulate_policies_workspace_bytes(dt: DeviceTrace, n_policies: int) -> int:
    tr = dt.c_struct()
    return int(lib().svf_simulate_policies_workspace_bytes(C.byref(tr), int(n_policies)))


def svf_simulate_policies(dt: DeviceTrace, policies, M: Optional[int] = None, outs=None,
                          ws: Optional[torch.Tensor] = None, want=RESULT_FIELDS, stream=None):
    """Enqueue the batched simulation under several policies in one call (one persistent launch
    over len(policies) x I work items); returns the list of SimOut, one per policy."""
    if not dt.offsets.is_cuda:
        raise TypeError("svf_simulate_policies needs device tensors (the library has no CPU path)")
    policies = [int(p) for p in policies]
    M = dt.M if M is None else int(M)
    if outs is None:
        outs = [SimOut.alloc(dt, want) for _ in policies]
    need = svf_simulate_policies_workspace_bytes(dt, len(policies))
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 256), dtype=torch.uint8, device=dt.offsets.device)
    tr = dt.c_struct()
    res = (_Result * len(policies))(*[o.c_struct() for o in outs])
    pol = (C.c_int * len(policies))(*policies)
    rc = lib().svf_simulate_policies(C.byref(tr), len(policies), pol, M, res, C.c_void_p(ws.data_ptr()),
                                     ws.numel(), _stream(stream))
    _check(rc, "svf_simulate_policies")
    _hold(ws, stream)
    for o in outs:
        o._ws = ws
    return outs


def svf_volume_lower_bound(dt: DeviceTrace, ws: Optional[torch.Tensor] = None, stream=None):
    """Prop. 3.1 lower bound per instance (int64 [I]) and its status (int32 [I])."""
    if not dt.offsets.is_cuda:
        raise TypeError("svf_volume_lower_bound needs device tensors (the library has no CPU path)")
    dev = dt.offsets.device
    tr = dt.c_struct()
    need = int(lib().svf_volume_lower_bound_workspace_bytes(C.byref(tr)))
    if ws is None or ws.numel() < need:
        ws = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    lb = torch.zeros(max(dt.n_instances, 1), dtype=torch.int64, device=dev)
    st = torch.zeros(max(dt.n_instances, 1), dtype=torch.int32, device=dev)
    rc = lib().svf_volume_lower_bound(C.byref(tr), C.c_void_p(lb.data_ptr()), C.c_void_p(st.data_ptr()),
                                      C.c_void_p(ws.data_ptr()), ws.numel(), _stream(stream))
    _check(rc, "svf_volume_lower_bound")
    _hold(ws, stream)
    return lb[: dt.n_instances], st[: dt.n_instances]
