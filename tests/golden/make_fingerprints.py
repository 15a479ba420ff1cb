"""Writes tests/golden/fingerprints.txt: the FNV-1a-64 fingerprint (traces.trace_fingerprint) of the
input arrays of every BASELINE.json config at its stated size.  Calls only the seeded input
generators (paper_2606_22327_b200/traces.py: numpy, none of the method's arithmetic); neither the
oracle nor the CUDA path is involved.  The generated ARRAYS are the contract between the two
(SURVEY 8(d)): a change of the generator that moves any element changes a line here.

    python tests/golden/make_fingerprints.py > tests/golden/fingerprints.txt
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_22327_b200 import traces as T  # noqa: E402


def cases():
    yield "configs[0] seed 0", T.config1(0)
    yield "configs[0] 512 seeds", T.concat([T.config1(i) for i in range(512)], "cfg1x512", 32, 2, 8)
    yield "configs[1] instance 0", T.config2(0)
    for lam in (2.0, 4.0, 8.0):
        yield f"configs[2] rate {lam:g}", T.config3(n_instances=4096, lam=lam)
    yield "configs[3]", T.config4()
    for M in (50_000, 200_000, 800_000):
        for p in (0.0, 0.05, 0.2):
            yield f"configs[4] M={M} p={p:g}", T.config5(M=M, p_flip=p)
    yield "stochastic rate 0.5 theta 293", T.stochastic(n_instances=64, n=1000, lam=0.5)


if __name__ == "__main__":
    print("# name | instances | requests | request_steps | fingerprint_fnv1a64   (written by make_fingerprints.py)")
    for name, tr in cases():
        print(f"{name} | {tr.n_instances} | {tr.n_requests} | {tr.request_steps} | {T.trace_fingerprint(tr)}")
