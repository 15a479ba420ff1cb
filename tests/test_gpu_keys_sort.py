"""GPU parity (bit-exact): svf_keys and the onesweep radix sort against the CPU oracle / numpy.
Run on the B200 box with ``-m gpu``; everything goes through the C ABI."""
import numpy as np
import pytest

from paper_2606_22327_b200 import traces as T

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_22327_b200 import binding
    binding.lib()
    return binding


def _dev(x, dt=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    return t if dt is None else t.to(dt)


def _u64(t):
    return t.cpu().numpy().view(np.uint64)


def _rand_requests(seed, n, s_hi=8192, o_hi=4096, a_hi=100000):
    sd = T.instance_seed(77, seed)
    s = T.uniform_int(sd, 2, n, 0, s_hi)
    o = T.uniform_int(sd, 4, n, 1, o_hi)
    a = np.sort(T.uniform_int(sd, 1, n, 0, a_hi))
    bit = (T.uniform(sd, 7, n) < 0.3).astype(np.uint8)
    return s, o, a, bit


@pytest.mark.parametrize("n", [0, 1, 3, 4, 5, 1023, 4097, (1 << 20) + 5])
@pytest.mark.parametrize("policy", [0, 1, 2, 3])
def test_keys_match_oracle(B, oracle, policy, n):
    s, o, a, bit = _rand_requests(n + policy, n)
    rc, want = oracle.keys(policy, s, o, a, bit, 179, 887)
    assert rc == 0
    words, status = B.svf_keys(policy, _dev(s), _dev(o), _dev(a), _dev(bit), 179, 887)
    assert int(status.item()) == 0
    assert np.array_equal(_u64(words), want)


def test_keys_unaligned_views_take_the_scalar_path(B, oracle):
    n = 10001
    s, o, a, bit = _rand_requests(5, n + 3)
    ds, do, da, db = _dev(s)[1:n + 1], _dev(o)[3:n + 3], _dev(a)[2:n + 2], _dev(bit)[1:n + 1]
    for policy in range(4):
        rc, want = oracle.keys(policy, s[1:n + 1], o[3:n + 3], a[2:n + 2], bit[1:n + 1], 5, 70)
        words, status = B.svf_keys(policy, ds, do, da, db, 5, 70)
        assert rc == 0 and int(status.item()) == 0
        assert np.array_equal(_u64(words), want)


def test_keys_16_byte_aligned_views_take_the_128_bit_path(B, oracle):
    """Arrays aligned to 16 but not to 32 bytes (and the words too): 128-bit accesses instead of the
    256-bit ones a fresh allocation gets; ragged sizes for both tails."""
    import torch
    for n in (10_000, 10_003, 7):
        s, o, a, bit = _rand_requests(6, n + 4)
        ds, do, da, db = _dev(s)[4:n + 4], _dev(o)[4:n + 4], _dev(a)[4:n + 4], _dev(bit)[4:n + 4]
        assert ds.data_ptr() % 32 == 16 and db.data_ptr() % 8 == 4
        buf = torch.empty(n + 2, dtype=torch.int64, device="cuda")
        for policy in range(4):
            rc, want = oracle.keys(policy, s[4:n + 4], o[4:n + 4], a[4:n + 4], bit[4:n + 4], 5, 70)
            words, status = B.svf_keys(policy, ds, do, da, db, 5, 70, words_out=buf[2:n + 2])
            assert rc == 0 and int(status.item()) == 0
            assert np.array_equal(_u64(words), want)


def test_keys_overflow_is_reported(B, oracle):
    s = np.array([1, 65536, 7, 9, 2], np.int32)
    o = np.array([1, 65536, 7, 9, 3], np.int32)
    rc, want = oracle.keys(0, s, o)
    assert rc == oracle.EOVERFLOW
    words, status = B.svf_keys(0, _dev(s), _dev(o))
    assert int(status.item()) == B.EOVERFLOW
    ok = np.array([0, 2, 3, 4])
    assert np.array_equal(_u64(words)[ok], want[ok])
    # paper limits: s <= 65536, o <= 4096 stay below 2^29
    s = np.array([65536], np.int32); o = np.array([4096], np.int32)
    words, status = B.svf_keys(0, _dev(s), _dev(o))
    assert int(status.item()) == 0 and int(_u64(words)[0] >> np.uint64(32)) == 65536 * 4096 + 4096 * 4097 // 2


def _stable_sort_on_bits(w, lo, hi):
    mask = np.uint64(((1 << (hi - lo)) - 1))
    k = (w >> np.uint64(lo)) & mask
    return w[np.argsort(k, kind="stable")]


@pytest.mark.parametrize("n", [0, 1, 2, 4095, 4096, 4097, 8192 + 17, (1 << 20) + 3])
@pytest.mark.parametrize("bits", [(0, 64), (32, 64), (10, 47), (5, 6), (0, 32), (13, 21)])
def test_sort_is_the_stable_sort_on_the_bit_range(B, n, bits):
    lo, hi = bits
    w = T.u64(T.instance_seed(55, n), 3, n)
    got = _u64(B.svf_sort_words(_dev(w.view(np.int64)), lo, hi))
    assert np.array_equal(got, _stable_sort_on_bits(w, lo, hi))


def test_sort_skips_constant_digits_and_keeps_order(B):
    n = 100_003
    r = T.u64(T.instance_seed(56, 0), 3, n)
    # keys < 2^20 in bits [32, 52): the two top digit passes are constant and skipped on device
    w = ((r % np.uint64(1 << 20)) << np.uint64(32)) | np.arange(n, dtype=np.uint64)
    got = _u64(B.svf_sort_words(_dev(w.view(np.int64)), 32, 64))
    assert np.array_equal(got, np.sort(w))
    # all words equal on the range: nothing runs, output = input
    w2 = (np.uint64(5) << np.uint64(32)) | np.arange(n, dtype=np.uint64)[::-1].copy()
    got2 = _u64(B.svf_sort_words(_dev(w2.view(np.int64)), 32, 64))
    assert np.array_equal(got2, w2)
    # already sorted and reverse sorted inputs
    w3 = np.sort(w)
    assert np.array_equal(_u64(B.svf_sort_words(_dev(w3.view(np.int64)), 0, 64)), w3)
    assert np.array_equal(_u64(B.svf_sort_words(_dev(w3[::-1].copy().view(np.int64)), 0, 64)), w3)


def test_keys_then_sort_gives_the_priority_order(B, oracle):
    """a1-a3 chained: ascending packed words == (key, arrival, id) order of the oracle's queue."""
    tr = T.config4(n=50_000)
    for policy in range(4):
        words, _ = B.svf_keys(policy, _dev(tr.prompt), _dev(tr.output), _dev(tr.arrival), _dev(tr.bit), tr.O0, tr.O1)
        got = _u64(B.svf_sort_words(words, 32, 64))
        rc, w = oracle.keys(policy, tr.prompt, tr.output, tr.arrival, tr.bit, tr.O0, tr.O1)
        assert rc == 0 and np.array_equal(got, np.sort(w))
