"""Pins for the NEXT-2 oracle functions (CPU only): delay-mode straggler (
DESIGN.md R19) and the model-disagreement diagnostic (eq. (9))."""
import numpy as np
import pytest

import oracle


def test_delay_straggler_is_active_every_nplus1_rounds():
    K, r, n = 8, 3, 4
    for t in range(40):
        _, act = oracle.schedule(7, t, 2, K, 0, 0.0, delay_replica=r, delay_rounds=n)
        want = np.ones(K, dtype=np.uint8)
        want[r] = 1 if (t + 1) % (n + 1) == 0 else 0          # one iteration per n+1 rounds
        assert np.array_equal(act, want)
    # off when delay_rounds == 0; combined with the random mask by AND
    assert all(oracle.active(7, t, r, 0.0, r, 0) == 1 for t in range(10))
    for t in range(200):
        a_rand = oracle.active(7, t, r, 0.5)
        a_both = oracle.active(7, t, r, 0.5, r, 1)
        assert a_both == (a_rand if (t + 1) % 2 == 0 else 0)


def test_delay_straggler_keeps_receiving_and_lags():
    """'The straggler keeps receiving updates from faster devices'; it performs
    1/(n+1) of the iterations: momentum changes only in its active rounds, weight never halves
    in between, x moves only through pushes while idle."""
    rng = np.random.default_rng(0)
    K, n_el, r, n = 6, 40, 2, 3
    o = oracle.Oracle([n_el], K, lr=0.01, momentum=0.9, seed=5, delay_replica=r, delay_rounds=n)
    o.x[0][:] = rng.normal(0, 0.02, (K, n_el)).astype(np.float32)
    own_steps = recv_idle = 0
    for t in range(48):
        peers, act = oracle.schedule(5, t, 1, K, 0, 0.0, delay_replica=r, delay_rounds=n)
        xb, mb, wb = o.x[0][r].copy(), o.m[0][r].copy(), o.w[0][r]
        o.round(t, [rng.normal(0, 1e-2, (K, n_el)).astype(np.float32)])
        senders = [s for s in range(K) if act[s] and peers[0][s] == r]
        if act[r]:
            own_steps += 1
            assert not np.array_equal(o.m[0][r], mb)
        else:
            assert np.array_equal(o.m[0][r], mb)
            assert o.w[0][r] >= wb                             # never halved while idle
            if senders:
                recv_idle += 1
                assert not np.array_equal(o.x[0][r], xb)
            else:
                assert np.array_equal(o.x[0][r], xb)
        assert abs(o.w[0].sum() - 1.0) < 1e-15
    assert own_steps == 48 // (n + 1) and recv_idle > 0


@pytest.mark.parametrize("weighted", [False, True])
def test_disagreement_against_numpy_and_identities(weighted):
    rng = np.random.default_rng(1)
    for K, n in [(2, 5), (3, 17), (8, 1000), (16, 33)]:
        x = rng.normal(0, 1, (K, n)).astype(np.float32)
        w = rng.dirichlet(np.ones(K)) if weighted else None
        c = w if weighted else np.full(K, 1.0 / K)
        got = oracle.disagreement(x, w)
        xd = x.astype(np.float64)
        xbar = (c[:, None] * xd).sum(0)
        want = ((xd - xbar[None, :]) ** 2).sum(1)              # independent numpy statement
        np.testing.assert_allclose(got, want, rtol=1e-12)
        # variance decomposition: sum_i c_i d_i = sum_i c_i ||x_i||^2 - ||xbar||^2
        lhs = (c * got).sum()
        rhs = (c * (xd ** 2).sum(1)).sum() - (xbar ** 2).sum()
        assert abs(lhs - rhs) <= 1e-10 * (c * (xd ** 2).sum(1)).sum()
        # translation invariance and quadratic scaling
        shift = rng.normal(0, 1, n)
        np.testing.assert_allclose(oracle.disagreement((xd + shift).astype(np.float32), w), got, rtol=1e-4, atol=1e-4)
        np.testing.assert_allclose(oracle.disagreement((2 * x).astype(np.float32), w), 4 * got, rtol=1e-12)


def test_disagreement_closed_forms():
    rng = np.random.default_rng(2)
    x = np.repeat(rng.normal(0, 1, (1, 50)).astype(np.float32), 5, 0)
    assert (oracle.disagreement(x) < 1e-28).all()                              # consensus: 0 up to fp64 rounding of 1/5
    assert np.array_equal(oracle.disagreement(x[:4]), np.zeros(4))             # 1/4 is exact: exactly 0
    a, b = rng.normal(0, 1, (2, 64)).astype(np.float32)
    d2 = ((a.astype(np.float64) - b) ** 2).sum()
    np.testing.assert_allclose(oracle.disagreement(np.stack([a, b])), [d2 / 4, d2 / 4], rtol=1e-12)   # K=2
    w = np.array([0.25, 0.75])
    np.testing.assert_allclose(oracle.disagreement(np.stack([a, b]), w), [d2 * 0.5625, d2 * 0.0625], rtol=1e-12)


def test_gossip_shrinks_disagreement_and_eq9_scaling():
    """Pure mixing drives every replica's distance to the weighted consensus to 0; with gradients
    of scale eta the stationary disagreement scales like eta^2 (eq. (9): <= eta^2 B^2)."""
    rng = np.random.default_rng(3)
    K, n = 8, 200
    o = oracle.Oracle([n], K, lr=0.0, momentum=0.0, seed=9)
    o.x[0][:] = rng.normal(0, 1, (K, n)).astype(np.float32)
    d0 = o.disagreement(weighted=True)[0]
    for t in range(80):
        o.round(t, [np.zeros((K, n), dtype=np.float32)])
    assert (o.disagreement(weighted=True)[0] < 1e-9 * d0.max()).all()
    tails = []
    for lr in (0.1, 0.01):
        o = oracle.Oracle([n], K, lr=lr, momentum=0.0, seed=9)
        acc = []
        for t in range(300):
            o.round(t, [rng.normal(0, 1, (K, n)).astype(np.float32)])
            if t >= 100:
                acc.append(o.disagreement()[0].mean())
        tails.append(np.mean(acc))
    assert 50 < tails[0] / tails[1] < 200                                       # ~ (0.1/0.01)^2 = 100
