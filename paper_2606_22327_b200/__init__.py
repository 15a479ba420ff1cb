"""B200-native hot path of "Geometry-Aware Online Scheduling for LLM Serving"
(arxiv/paper_2606_22327): SVF / 1-bit SVF admission inside a batched discrete-time simulator of
the paper's KV-cache memory model, as hand-written sm_100a CUDA kernels behind a C ABI
(``svf_keys``, ``svf_admit``, ``svf_simulate``; see ``include/svf.h``).

``traces``  -- seeded synthetic input generators (numpy only; shared with the oracle's tests).
``binding`` -- thin ctypes binding over ``csrc/libsvf_b200.so`` (argument marshalling only).
The binding is imported lazily so that ``traces`` stays usable without the CUDA library.
"""

__all__ = ["traces", "binding"]


def __getattr__(name):
    if name in ("traces", "binding"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)
