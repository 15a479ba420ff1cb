"""Seeded synthetic trace generators for the five BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA path: it
produces the input arrays ``(offsets, arrival, prompt, output, bit)`` plus the scalars
``(M, O0, O1)`` and holds none of the method's arithmetic (no keys, no feasibility, no
simulation).  numpy only; it never imports the binding or the oracle.

The traces stand in for the paper's LMSYS-Chat-1M / LongBench / BurstGPT workloads
(PAPER.md:211, :237), none of which is available here; shapes, rates and length laws are the
ones BASELINE.json's ``configs`` give, with the readings R14/R15 of SURVEY.md §8(c) (recipe
restated in DESIGN.md §4).

Generator: counter based.  ``u64(seed, stream, i) = mix(mix(seed ^ stream*C1) + i*C2)`` with
``mix`` the splitmix64 finaliser; uniform double ``(u >> 11) * 2**-53``; normal deviates by
Box-Muller; exponential gaps ``-ln(1-u)/lambda`` accumulated in double and floored.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 260622327

_C1 = np.uint64(0x9E3779B97F4A7C15)
_C2 = np.uint64(0xD1342543DE82EF95)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

# stream ids (one independent sequence per quantity)
_ST_GAP, _ST_S1, _ST_S2, _ST_O1, _ST_O2, _ST_MODE, _ST_FLIP, _ST_SEED = range(1, 9)


def _mix(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        x = np.asarray(x, dtype=np.uint64).copy()
        x ^= x >> np.uint64(30)
        x *= _M1
        x ^= x >> np.uint64(27)
        x *= _M2
        x ^= x >> np.uint64(31)
    return x


def u64(seed: int, stream: int, n: int) -> np.ndarray:
    """n counter-based 64-bit draws of stream ``stream`` under ``seed``."""
    with np.errstate(over="ignore"):
        k0 = (seed ^ (stream * int(_C1))) & 0xFFFFFFFFFFFFFFFF
        k = _mix(np.array([k0], dtype=np.uint64))
        idx = np.arange(n, dtype=np.uint64)
        return _mix(k + (idx + np.uint64(1)) * _C2)


def uniform(seed: int, stream: int, n: int) -> np.ndarray:
    """Uniform doubles in [0, 1)."""
    return (u64(seed, stream, n) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def uniform_int(seed: int, stream: int, n: int, lo: int, hi: int) -> np.ndarray:
    """Uniform integers in {lo..hi} (inclusive)."""
    u = uniform(seed, stream, n)
    return (lo + np.floor(u * (hi - lo + 1))).astype(np.int64).clip(lo, hi).astype(np.int32)


def normal(seed: int, st1: int, st2: int, n: int) -> np.ndarray:
    """Standard normal deviates (Box-Muller, cosine branch)."""
    u1 = 1.0 - uniform(seed, st1, n)           # (0, 1]
    u2 = uniform(seed, st2, n)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


def lognormal_int(seed: int, st1: int, st2: int, n: int, mean: float, sigma: float,
                  lo: int, hi: int) -> np.ndarray:
    """clip(rint(exp(mu + sigma z)), lo, hi) with mu = ln(mean) - sigma^2/2:
    ``mean`` is the arithmetic mean of the unclipped law."""
    mu = math.log(mean) - 0.5 * sigma * sigma
    v = np.exp(mu + sigma * normal(seed, st1, st2, n))
    return np.clip(np.rint(v), lo, hi).astype(np.int32)


def poisson_arrivals(seed: int, n: int, lam: float) -> np.ndarray:
    """Arrival steps of a rate-``lam`` Poisson process: exponential gaps summed in
    double, floored to an integer step.  Non-decreasing by construction."""
    gaps = -np.log(1.0 - uniform(seed, _ST_GAP, n)) / lam
    return np.floor(np.cumsum(gaps)).astype(np.int32)


def instance_seed(config: int, instance: int, variant: int = 0) -> int:
    s = (BASE_SEED + 1000 * config + instance + 7919 * 1000003 * variant) & 0xFFFFFFFFFFFFFFFF
    s ^= (_ST_SEED * int(_C1)) & 0xFFFFFFFFFFFFFFFF
    return int(_mix(np.array([s], dtype=np.uint64))[0])


@dataclass
class Trace:
    """A batch of independent instances in the layout the C ABI takes (SoA, instances
    concatenated; ``offsets[j]:offsets[j+1]`` is instance j, arrivals non-decreasing inside)."""
    name: str
    offsets: np.ndarray      # int64 [I+1]
    arrival: np.ndarray      # int32 [N]
    prompt: np.ndarray       # int32 [N]
    output: np.ndarray       # int32 [N]
    bit: np.ndarray          # uint8 [N]
    M: int
    O0: int
    O1: int
    meta: dict = field(default_factory=dict)
    output_key: np.ndarray = None   # int32 [N] predicted output lengths (key only) or None

    @property
    def n_instances(self) -> int:
        return len(self.offsets) - 1

    @property
    def n_requests(self) -> int:
        return int(self.offsets[-1])

    @property
    def max_n(self) -> int:
        return int(np.max(np.diff(self.offsets))) if self.n_instances else 0

    @property
    def request_steps(self) -> int:
        """sum_i o_i: the policy-independent work measure of SURVEY §8(d)."""
        return int(self.output.astype(np.int64).sum())

    def instance(self, j: int) -> "Trace":
        lo, hi = int(self.offsets[j]), int(self.offsets[j + 1])
        return Trace(f"{self.name}[{j}]", np.array([0, hi - lo], dtype=np.int64),
                     self.arrival[lo:hi].copy(), self.prompt[lo:hi].copy(),
                     self.output[lo:hi].copy(), self.bit[lo:hi].copy(), self.M, self.O0, self.O1,
                     dict(self.meta),
                     None if self.output_key is None else self.output_key[lo:hi].copy())

    def subset(self, idx) -> "Trace":
        parts = [self.instance(int(j)) for j in idx]
        return concat(parts, self.name + "[subset]", self.M, self.O0, self.O1, dict(self.meta))

    def checksum(self) -> int:
        """Order-sensitive 64-bit checksum of the input arrays (identity of the inputs):
        xor-fold of mix(value_i + (i+1)*C2 + array_tag*C1), vectorised."""
        h = np.uint64(0)
        with np.errstate(over="ignore"):
            for tag, arr in enumerate((self.offsets, self.arrival, self.prompt, self.output,
                                       self.bit), start=1):
                v = np.ascontiguousarray(arr).astype(np.int64).view(np.uint64)
                idx = np.arange(1, len(v) + 1, dtype=np.uint64)
                m = _mix(v + idx * _C2 + np.uint64(tag) * _C1)
                h ^= np.bitwise_xor.reduce(m) if len(m) else np.uint64(0)
                h = _mix(np.array([h]))[0]
        return int(h)


def fnv1a64(data: bytes) -> int:
    """FNV-1a, 64 bit, over a byte string (offset basis 0xcbf29ce484222325, prime 0x100000001b3)."""
    h = 0xCBF29CE484222325
    for b in data:
        h = ((h ^ b) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
    return h


def trace_fingerprint(tr: "Trace") -> str:
    """The identity of a config's input arrays as printed by bench.py: FNV-1a-64 (hex) over the
    little-endian bytes of (I, N, M, O0, O1, Trace.checksum()) -- the checksum folds every element of
    offsets / arrival / prompt / output / bit with its position, so the 48 bytes pin all of them.
    (FNV itself is sequential byte by byte: the large arrays go through the vectorised fold first.)"""
    words = np.array([tr.n_instances, tr.n_requests, tr.M, tr.O0, tr.O1], dtype=np.int64).view(np.uint64)
    words = np.concatenate([words, np.array([tr.checksum()], dtype=np.uint64)])
    return f"{fnv1a64(words.astype('<u8').tobytes()):016x}"


def admit_state(seed: int, n_wait: int, n_run: int, M: int, fill: float = 0.8):
    """Inputs of one stateless admission decision (bench.py's svf_admit sweep; BASELINE.json configs[3]
    laws for the waiting queue): waiting (s, o, a, bit) in arrival order and a running set (kv, rem)
    with uniform remaining steps and lognormal held tokens, the tokens scaled down so that the final
    footprints sum to at most ``fill * M``:  sum_j (kv_j + rem_j) <= fill * M.  A request never holds
    more than kv + rem, so the set is feasible on its own whatever the order of completions -- a loaded
    engine with room for a few more.  Input shaping only (two sums of the generator's own draws):
    no key, no ordering by completion time, no feasibility check."""
    sd = instance_seed(88, seed)
    w_s = lognormal_int(sd, 2, 3, n_wait, 1000.0, 0.8, 16, 8192)
    w_o = lognormal_int(sd, 4, 5, n_wait, 400.0, 1.0, 1, 4096)
    w_a = np.sort(uniform_int(sd, 1, n_wait, 0, 5000))
    w_bit = (w_o > 400).astype(np.uint8)
    rem_hi = int(max(8, min(3000, fill * M / max(n_run, 1))))      # mean rem = half of an equal share of fill * M
    r_rem = uniform_int(sd, 6, n_run, 1, rem_hi)
    r_kv = lognormal_int(sd, 7, 8, n_run, 1200.0, 0.8, 16, 12000)
    if n_run:
        room = fill * M - float(r_rem.astype(np.int64).sum())
        scale = float(np.clip(room / float(r_kv.astype(np.int64).sum()), 0.0, 1.0))
        r_kv = np.maximum((r_kv * scale).astype(np.int32), 0)
    return w_s, w_o, w_a, w_bit, r_kv, r_rem


def concat(parts, name, M, O0, O1, meta=None) -> Trace:
    sizes = [p.n_requests for p in parts]
    offsets = np.zeros(len(parts) + 1, dtype=np.int64)
    offsets[1:] = np.cumsum(sizes)
    cat = lambda key, dt: (np.concatenate([getattr(p, key) for p in parts]).astype(dt)
                           if parts else np.zeros(0, dt))
    okey = None
    if parts and all(p.output_key is not None for p in parts):
        okey = cat("output_key", np.int32)
    return Trace(name, offsets, cat("arrival", np.int32), cat("prompt", np.int32),
                 cat("output", np.int32), cat("bit", np.uint8), M, O0, O1, meta or {}, okey)


def _one(name, a, s, o, bit, M, O0, O1, meta=None) -> Trace:
    n = len(a)
    return Trace(name, np.array([0, n], dtype=np.int64), a.astype(np.int32), s.astype(np.int32),
                 o.astype(np.int32), bit.astype(np.uint8), int(M), int(O0), int(O1), meta or {})


# ---------------------------------------------------------------------------------------------
# Config 1: tiny offline instance (BASELINE.json configs[0])
# ---------------------------------------------------------------------------------------------
def config1(instance: int = 0, n: int = 8, M: int = 32, hi: int = 8) -> Trace:
    """n requests at t=0, s,o ~ U{1..hi}, M tokens.  bit = (o_i > median), the median of an even
    sample compared in doubled integers.  O0=2, O1=8: the Thm 3.3 recipe
     at T=16=max(s+o): theta=4, O0=T^(1/4), O1=T^(3/4)."""
    sd = instance_seed(1, instance)
    s = uniform_int(sd, _ST_S1, n, 1, hi)
    o = uniform_int(sd, _ST_O1, n, 1, hi)
    so = np.sort(o.astype(np.int64))
    med2 = so[(n - 1) // 2] + so[n // 2]          # twice the median
    bit = (2 * o.astype(np.int64) > med2).astype(np.uint8)
    return _one(f"cfg1[{instance}]", np.zeros(n, np.int32), s, o, bit, M, 2, 8,
                {"config": 1, "burst": True})


# ---------------------------------------------------------------------------------------------
# Config 2/3: online traces with lognormal lengths (configs[1], configs[2])
# ---------------------------------------------------------------------------------------------
def _online_lognormal(sd: int, n: int, lam: float, s_mean: float, s_sigma: float, s_lo: int,
                      s_hi: int, o_mean: float, o_sigma: float, o_lo: int, o_hi: int):
    a = poisson_arrivals(sd, n, lam)
    s = lognormal_int(sd, _ST_S1, _ST_S2, n, s_mean, s_sigma, s_lo, s_hi)
    o = lognormal_int(sd, _ST_O1, _ST_O2, n, o_mean, o_sigma, o_lo, o_hi)
    return a, s, o


# class-conditional proxies for lognormal outputs (mean 250, sigma 1, clip [1, 2048]) split at
# theta = 256 tokens (the rounded sample class means of this generator): harness constants in
# the spirit of Thm 3.5 (conditional-expectation proxies), not the paper's values.
LN_THETA, LN_O0, LN_O1 = 256, 113, 572


def config2(instance: int = 0, n: int = 2000, lam: float = 4.0, M: int = 300_000) -> Trace:
    sd = instance_seed(2, instance)
    a, s, o = _online_lognormal(sd, n, lam, 600.0, 0.8, 16, 4096, 250.0, 1.0, 1, 2048)
    bit = (o > LN_THETA).astype(np.uint8)
    return _one(f"cfg2[{instance}]", a, s, o, bit, M, LN_O0, LN_O1, {"config": 2, "lam": lam})


def config3(n_instances: int = 4096, n: int = 1000, lam: float = 4.0, M: int = 300_000,
            first_instance: int = 0) -> Trace:
    lam_tag = int(round(lam * 16))
    parts = []
    for j in range(first_instance, first_instance + n_instances):
        sd = instance_seed(3, j, variant=lam_tag)
        a, s, o = _online_lognormal(sd, n, lam, 600.0, 0.8, 16, 4096, 250.0, 1.0, 1, 2048)
        parts.append(_one("", a, s, o, (o > LN_THETA).astype(np.uint8), M, LN_O0, LN_O1))
    return concat(parts, f"cfg3[lam={lam:g}]", M, LN_O0, LN_O1, {"config": 3, "lam": lam})


# ---------------------------------------------------------------------------------------------
# Config 4: high-concurrency single instance (configs[3])
# ---------------------------------------------------------------------------------------------
C4_THETA, C4_O0, C4_O1 = 400, 179, 887


def config4(instance: int = 0, n: int = 200_000, lam: float = 64.0, M: int = 1_000_000) -> Trace:
    sd = instance_seed(4, instance)
    a, s, o = _online_lognormal(sd, n, lam, 1000.0, 0.8, 16, 8192, 400.0, 1.0, 1, 4096)
    bit = (o > C4_THETA).astype(np.uint8)
    return _one(f"cfg4[{instance}]", a, s, o, bit, M, C4_O0, C4_O1, {"config": 4, "lam": lam})


# ---------------------------------------------------------------------------------------------
# Config 5: 1-bit SVF sweep (configs[4])
# ---------------------------------------------------------------------------------------------
def config5(n_instances: int = 256, n: int = 5000, M: int = 200_000, p_flip: float = 0.0,
            lam: float = 4.0, first_instance: int = 0) -> Trace:
    """Bimodal outputs: 70% U{8..128}, 30% U{512..2048}; prompts and arrivals as config 2
    (SURVEY R15).  True bit = (o >= 512), flipped with probability ``p_flip``.  O0=68, O1=1280
    are the class means of the generating law."""
    parts = []
    for j in range(first_instance, first_instance + n_instances):
        sd = instance_seed(5, j)
        a = poisson_arrivals(sd, n, lam)
        s = lognormal_int(sd, _ST_S1, _ST_S2, n, 600.0, 0.8, 16, 4096)
        mode = uniform(sd, _ST_MODE, n) < 0.7
        o_short = uniform_int(sd, _ST_O1, n, 8, 128)
        o_long = uniform_int(sd, _ST_O2, n, 512, 2048)
        o = np.where(mode, o_short, o_long).astype(np.int32)
        flip = uniform(sd, _ST_FLIP, n) < p_flip
        bit = ((o >= 512) ^ flip).astype(np.uint8)
        parts.append(_one("", a, s, o, bit, M, 68, 1280))
    return concat(parts, f"cfg5[M={M},p={p_flip:g}]", M, 68, 1280,
                  {"config": 5, "lam": lam, "p_flip": p_flip})


# ---------------------------------------------------------------------------------------------
# Free-form random instances for property tests (not one of the five configs)
# ---------------------------------------------------------------------------------------------
def random_small(seed: int, n: int, s_hi: int, o_hi: int, M: int, a_hi: int = 0,
                 O0: int = 2, O1: int = 8) -> Trace:
    """n requests, s ~ U{0..s_hi}, o ~ U{1..o_hi}, arrivals sorted U{0..a_hi}; every request is
    individually feasible if s_hi + o_hi <= M."""
    sd = instance_seed(99, seed)
    s = uniform_int(sd, _ST_S1, n, 0, s_hi)
    o = uniform_int(sd, _ST_O1, n, 1, o_hi)
    a = np.sort(uniform_int(sd, _ST_GAP, n, 0, a_hi)) if a_hi > 0 else np.zeros(n, np.int32)
    bit = (uniform(sd, _ST_FLIP, n) < 0.5).astype(np.uint8)
    return _one(f"rand[{seed}]", a, s, o, bit, M, O0, O1, {"burst": a_hi == 0})


# ---------------------------------------------------------------------------------------------
# Predicted output lengths: a stand-in for the paper's BERT length predictor
# (PAPER.md:215), which needs prompts and trained weights that are not available here
# ---------------------------------------------------------------------------------------------
def with_predicted_lengths(trace: Trace, sigma: float = 0.5, seed: int = 0, hi: int = 1 << 20) -> Trace:
    """A copy of ``trace`` with ``output_key[i] = clip(rint(o_i * exp(sigma * z_i)), 1, hi)``,
    z_i standard normal from the counter-based generator: multiplicative lognormal prediction
    noise (sigma = 0 reproduces the true lengths).  Only the ORDER of SVF / SJF sees it."""
    sd = instance_seed(77, seed)
    n = trace.n_requests
    z = normal(sd, _ST_O1, _ST_O2, n)
    ok = np.clip(np.rint(trace.output.astype(np.float64) * np.exp(sigma * z)), 1, hi).astype(np.int32)
    return Trace(trace.name + f"[pred sigma={sigma:g}]", trace.offsets.copy(), trace.arrival.copy(),
                 trace.prompt.copy(), trace.output.copy(), trace.bit.copy(), trace.M, trace.O0, trace.O1,
                 dict(trace.meta), ok)


# ---------------------------------------------------------------------------------------------
# Stochastic-regime workload: the paper's reference model of App. H
# (PAPER.md:866-870): Poisson arrivals, o ~ Geo(mu) truncated at the generation budget
# ---------------------------------------------------------------------------------------------
def geometric_int(seed: int, stream: int, n: int, mu: float, hi: int) -> np.ndarray:
    """o = min(hi, 1 + floor(ln(1-u) / ln(1-mu))): Pr(o = k) = mu (1-mu)^(k-1) on {1, 2, ..}
    (inverse CDF), truncated at ``hi`` (the paper's "maximum generation budget")."""
    u = uniform(seed, stream, n)
    k = 1 + np.floor(np.log1p(-u) / math.log1p(-mu))
    return np.clip(k, 1, hi).astype(np.int32)


def onebit_proxies(mu: float, theta: int):
    """Thm 3.5's proxy lengths for threshold theta under Geo(mu), rounded to integers >= 1
    (reading R9): O0 = 1/mu - theta q^theta / (1 - q^theta) (short: o <= theta), O1 = theta + 1/mu (long)."""
    q_t = (1.0 - mu) ** theta
    O0 = max(1, int(round(1.0 / mu - theta * q_t / (1.0 - q_t))))
    O1 = max(1, int(round(theta + 1.0 / mu)))
    return O0, O1


def stochastic(n_instances: int = 64, n: int = 1000, lam: float = 1.0, mean_o: float = 293.0,
               o_hi: int = 4096, M: int = 300_000, first_instance: int = 0, theta: int = None) -> Trace:
    """Poisson(lam) arrivals, o ~ Geo(1/mean_o) truncated at o_hi (mean 293 and budget 4,096 are the
    paper's calibration), prompts as config 2.  1-bit constants follow Thm 3.5's
    conditional-expectation recipe at theta = mean_o, rounded to integers:
    O0 = 1/mu - theta q^theta / (1 - q^theta), O1 = theta + 1/mu, q = 1 - mu."""
    mu = 1.0 / mean_o
    theta = int(round(mean_o)) if theta is None else int(theta)      # the 1-bit threshold: bit = (o > theta)
    O0, O1 = onebit_proxies(mu, theta)
    parts = []
    for j in range(first_instance, first_instance + n_instances):
        sd = instance_seed(6, j, variant=int(round(lam * 16)))
        a = poisson_arrivals(sd, n, lam)
        s = lognormal_int(sd, _ST_S1, _ST_S2, n, 600.0, 0.8, 16, 4096)
        o = geometric_int(sd, _ST_O1, n, mu, o_hi)
        parts.append(_one("", a, s, o, (o > theta).astype(np.uint8), M, O0, O1))
    return concat(parts, f"geo[lam={lam:g},1/mu={mean_o:g},theta={theta}]", M, O0, O1,
                  {"config": 6, "lam": lam, "mu": mu, "theta": theta})
