"""Pins for the oracle's Philox4x32-10 and for the schedule it drives (CPU only).

Pin (i): cuRAND's library routine curand_Philox4x32_10, compiled for the host by
tests/curand_pin.cpp -- an implementation that is not ours.  Pins (ii): the properties
PAPER.md:101,106 fix: the peer is never the worker itself, it is uniform over the other
M-1 workers, and the skip rate matches the requested probability.
"""
import numpy as np
import pytest

import oracle


def _curand(lib, ctr, key):
    out = np.empty_like(ctr)
    lib.curand_philox_host(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, ctr.shape[0])
    return out


def test_philox_matches_curand_library(curand_pin):
    rng = np.random.default_rng(1234)
    n = 200_000
    ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    # edge patterns: zeros, all ones, single bits
    ctr[0] = 0; key[0] = 0
    ctr[1] = 0xFFFFFFFF; key[1] = 0xFFFFFFFF
    for b in range(32):
        ctr[2 + b] = 0; ctr[2 + b, b % 4] = np.uint32(1) << np.uint32(b); key[2 + b] = (b, 0)
    want = _curand(curand_pin, ctr, key)
    L = oracle.lib()
    got = np.empty_like(ctr)
    for i in range(n):
        L.oracle_philox4x32_10(ctr[i].ctypes.data, key[i].ctypes.data, got[i].ctypes.data)
    assert np.array_equal(got, want)


def test_peer_uses_first_word_of_keyed_counter(curand_pin):
    """peer = mulhi(philox(key=seed; step, layer, replica, 0).x, K-1) skipping self (DESIGN R5, R6)."""
    seed = 0x1234567_89ABCDEF
    for (step, layer, rep, K) in [(0, 0, 0, 2), (7, 3, 5, 8), (2**31, 146, 15, 16), (99, 39, 63, 64)]:
        ctr = np.array([[step & 0xFFFFFFFF, layer, rep, 0]], dtype=np.uint32)
        key = np.array([[seed & 0xFFFFFFFF, seed >> 32]], dtype=np.uint32)
        r = int(_curand(curand_pin, ctr, key)[0, 0])
        q = (r * (K - 1)) >> 32
        assert oracle.peer(seed, step, layer, rep, K, 0) == q + (1 if q >= rep else 0)
        # peer_mode 1 replaces the layer field by 0xFFFFFFFF: same peer for every layer
        ctr[0, 1] = 0xFFFFFFFF
        r = int(_curand(curand_pin, ctr, key)[0, 0])
        q = (r * (K - 1)) >> 32
        assert oracle.peer(seed, step, layer, rep, K, 1) == q + (1 if q >= rep else 0)
        assert oracle.peer(seed, step, layer, rep, K, 1) == oracle.peer(seed, step, layer + 1, rep, K, 1)


def test_skip_uses_tag_one_and_threshold(curand_pin):
    seed = 42
    for p in (0.25, 0.5, 0.9, 1.0):
        thr = min(int(float(np.float32(p)) * 4294967296.0), 0xFFFFFFFF)
        for step in range(20):
            for rep in range(8):
                ctr = np.array([[step, 0xFFFFFFFF, rep, 1]], dtype=np.uint32)
                key = np.array([[seed, 0]], dtype=np.uint32)
                r = int(_curand(curand_pin, ctr, key)[0, 0])
                assert oracle.active(seed, step, rep, p) == (0 if r < thr else 1)
    assert all(oracle.active(seed, s, r, 0.0) == 1 for s in range(10) for r in range(4))


@pytest.mark.parametrize("K", [2, 3, 4, 8, 16, 64])
def test_peer_never_self_and_uniform(K):
    """PAPER.md:101 Random(M-1), PAPER.md:106 'uniformly at random'."""
    steps, L = 400, 8
    counts = np.zeros((K, K), dtype=np.int64)
    for t in range(steps):
        p, a = oracle.schedule(5, t, L, K, 0, 0.0)
        assert a.all()
        assert ((p >= 0) & (p < K)).all()
        assert (p != np.arange(K)[None, :]).all()
        for i in range(K):
            counts[i] += np.bincount(p[:, i], minlength=K)
    n = steps * L
    if K > 2:
        exp = n / (K - 1)
        for i in range(K):
            obs = np.delete(counts[i], i)
            chi2 = ((obs - exp) ** 2 / exp).sum()
            # chi-square with K-2 dof: mean K-2, std sqrt(2(K-2)); 6-sigma gate
            assert chi2 < (K - 2) + 6 * np.sqrt(2 * (K - 2)) + 10, (i, chi2)
    else:
        assert counts[0, 1] == n and counts[1, 0] == n


def test_skip_rate_and_straggler_schedule():
    K, p = 8, 0.25
    act = np.array([oracle.schedule(3, t, 3, K, 0, p)[1] for t in range(4000)])
    rate = 1.0 - act.mean()
    assert abs(rate - p) < 4 * np.sqrt(p * (1 - p) / act.size)
    # an inactive replica has no peer in any layer of that round; active ones do
    for t in range(50):
        peer, a = oracle.schedule(3, t, 3, K, 0, p)
        assert ((peer >= 0) == a.astype(bool)[None, :]).all()


def test_schedule_depends_on_every_key_field():
    K, L = 16, 6
    base = oracle.schedule(9, 4, L, K, 0, 0.0)[0]
    assert not np.array_equal(base, oracle.schedule(10, 4, L, K, 0, 0.0)[0])       # seed
    assert not np.array_equal(base, oracle.schedule(9 + (1 << 32), 4, L, K, 0, 0.0)[0])  # seed high word
    assert not np.array_equal(base, oracle.schedule(9, 5, L, K, 0, 0.0)[0])        # step
    assert not np.array_equal(base[0], base[1])                                    # layer
    assert np.array_equal(base, oracle.schedule(9, 4, L, K, 0, 0.0)[0])            # pure function
    m1 = oracle.schedule(9, 4, L, K, 1, 0.0)[0]
    assert (m1 == m1[0][None, :]).all()                                            # Alg. 1: one peer per iteration
