"""The seeded input generators (paper_2606_22327_b200/traces.py): the arrays they produce are the
contract between the oracle and the CUDA path.  CPU only."""
import importlib.util
import os

import numpy as np

from paper_2606_22327_b200 import traces as T

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_fnv1a64_published_test_vectors():
    # the FNV-1a reference vectors: "" -> offset basis, "a", "foobar"
    assert T.fnv1a64(b"") == 0xCBF29CE484222325
    assert T.fnv1a64(b"a") == 0xAF63DC4C8601EC8C
    assert T.fnv1a64(b"foobar") == 0x85944171F73967E8


def test_fingerprints_of_every_config_match_the_stored_ones():
    """tests/golden/fingerprints.txt (written by make_fingerprints.py from the generators alone): any
    change of a generated element, of a size or of M / O0 / O1 moves a fingerprint."""
    spec = importlib.util.spec_from_file_location("make_fingerprints", os.path.join(GOLDEN, "make_fingerprints.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    want = {}
    for line in open(os.path.join(GOLDEN, "fingerprints.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, I, N, rs, fp = [x.strip() for x in line.split("|")]
        want[name] = (int(I), int(N), int(rs), fp)
    seen = 0
    for name, tr in mod.cases():
        assert (tr.n_instances, tr.n_requests, tr.request_steps, T.trace_fingerprint(tr)) == want[name], name
        seen += 1
    assert seen == len(want) >= 17


def test_fingerprint_sees_every_array_and_scalar():
    tr = T.config2(0, n=300)
    base = T.trace_fingerprint(tr)
    for field in ("arrival", "prompt", "output", "bit"):
        arr = getattr(tr, field)
        old = arr[17]
        arr[17] = old + 1
        assert T.trace_fingerprint(tr) != base, field
        arr[17] = old
    assert T.trace_fingerprint(tr) == base
    tr.M += 1
    assert T.trace_fingerprint(tr) != base


def test_config_shapes_and_laws():
    """Sizes, ranges and order of what BASELINE.json's configs state (recipe in DESIGN.md 4)."""
    c1 = T.config1(3)
    assert c1.n_requests == 8 and c1.M == 32 and not c1.arrival.any()
    assert c1.prompt.min() >= 1 and c1.prompt.max() <= 8 and c1.output.min() >= 1 and c1.output.max() <= 8
    c2 = T.config2(0)
    assert c2.n_requests == 2000 and c2.M == 300_000
    assert (np.diff(c2.arrival) >= 0).all() and 16 <= c2.prompt.min() and c2.prompt.max() <= 4096
    assert 1 <= c2.output.min() and c2.output.max() <= 2048
    assert abs(c2.arrival[-1] / 2000 - 0.25) < 0.03                    # Poisson rate 4 per step
    c4 = T.config4(n=20_000)
    assert c4.prompt.max() <= 8192 and c4.output.max() <= 4096 and abs(c4.arrival[-1] / 20_000 - 1 / 64) < 0.002
    c5 = T.config5(n_instances=4, p_flip=0.2)
    short = c5.output <= 128
    assert ((c5.output >= 8) & short | (c5.output >= 512) & (c5.output <= 2048)).all()
    assert abs(short.mean() - 0.7) < 0.02
    flipped = (c5.bit != (c5.output >= 512)).mean()
    assert abs(flipped - 0.2) < 0.02
    assert np.array_equal(T.config5(n_instances=4, p_flip=0.0).output, c5.output)      # p only touches the bits


def test_admit_state_is_a_loaded_but_feasible_engine():
    for W, R, M in ((1000, 256, 1_000_000), (100, 4096, 1_000_000), (50, 0, 10_000)):
        w_s, w_o, w_a, w_bit, r_kv, r_rem = T.admit_state(W + R, W, R, M)
        assert len(w_s) == W and len(r_kv) == R and (np.diff(w_a) >= 0).all()
        assert (r_rem >= 1).all() and (r_kv >= 0).all()
        if R:
            # the running set alone: memory at its completion times (latest finish first) stays under M
            order = np.argsort(-r_rem, kind="stable")
            peak = (np.cumsum(r_kv[order].astype(np.int64)) + r_rem[order].astype(np.int64) * np.arange(1, R + 1)).max()
            assert peak <= 0.8 * M + R
            # ... which the generator guarantees through the final footprints alone (no completion-time formula in it)
            assert int((r_kv.astype(np.int64) + r_rem).sum()) <= 0.8 * M or not r_kv.any()
