"""Pins for the oracle's update + gossip rule (CPU only): what the paper and the
mathematics fix, never the oracle's own formula re-typed.

W1-W3  hand-derived worked examples (tests/golden/, each citing PAPER.md)
I1     push-sum mass conservation, sum_i w_i = 1, E[w_i] = 1/M
I2     weighted-mean conservation under a pure mix
I3     K = 2 exact pairwise averaging                                   (north_star)
I4     weighted consensus distance non-increasing, -> 0
I5     convexity of the peer update
I6     brute force: every peer map x every active mask on tiny layers against a dense
       row-stochastic matrix product written independently in numpy fp64
I7     K = 1 reduces to torch.optim.SGD (textbook / library routine)
I8     consensus is a fixed point (bit-identical replicas stay bit-identical)
I9     layers are independent (any layer order gives the same bits)
I10    peer_mode 1 reproduces Algorithm 1's scalar w_i
"""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

import oracle

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _read_golden(name):
    d = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, *v = line.split()
            d[k] = [float(Fraction(t)) for t in v]
    return d


@pytest.mark.parametrize("name", ["W1_three_workers.txt", "W2_two_workers.txt", "W3_momentum_straggler.txt"])
def test_worked_examples(name):
    d = _read_golden(name)
    K = int(d["K"][0])
    lr = d.get("lr", [0.0])[0]
    mu = d.get("mu", [0.0])[0]
    x = np.array(d["x_before"], dtype=np.float32).reshape(K, 1)
    g = np.array(d.get("g", [0.0] * K), dtype=np.float32).reshape(K, 1)
    m = np.array(d.get("m_before", [0.0] * K), dtype=np.float32).reshape(K, 1)
    w = np.array(d["w_before"], dtype=np.float64)
    peer = np.array(d["peer"], dtype=np.int32)
    act = np.array(d.get("active", [1.0] * K), dtype=np.uint8)
    oracle.layer_update(x, g, m, w, lr, mu, 0, 0, 0, peer_in=peer, active_in=act)
    np.testing.assert_allclose(x[:, 0], d["x_after"], rtol=2e-7, atol=0)
    np.testing.assert_allclose(w, d["w_after"], rtol=1e-15, atol=0)
    if "m_after" in d:
        np.testing.assert_array_equal(m[:, 0], np.array(d["m_after"], dtype=np.float32))
    # the fp64 shadow is a second statement of the same rule (closed-form centroid)
    x64 = np.array(d["x_before"], dtype=np.float64).reshape(K, 1)
    m64 = np.array(d.get("m_before", [0.0] * K), dtype=np.float64).reshape(K, 1)
    w64 = np.array(d["w_before"], dtype=np.float64)
    oracle.layer_update(x64, g, m64, w64, lr, mu, 0, 0, 0, peer_in=peer, active_in=act)
    np.testing.assert_allclose(x64[:, 0], d["x_after"], rtol=1e-15)
    np.testing.assert_allclose(w64, d["w_after"], rtol=1e-15)


def test_k2_draws_the_other_worker_and_averages_exactly():
    """I3 / W2 with the peers drawn by the oracle itself, random representable values."""
    rng = np.random.default_rng(0)
    for step in range(20):
        # multiples of 2^-10 below 2^6: x0 + x1 and the halves are exact in fp32
        x = (rng.integers(-2**16, 2**16, size=(2, 257)) / 1024.0).astype(np.float32)
        want = ((x[0].astype(np.float64) + x[1]) / 2).astype(np.float32)
        g = np.zeros_like(x)
        w = np.array([0.5, 0.5])
        oracle.layer_update(x, g, None, w, 0.1, 0.0, 77, step, 0)
        assert np.array_equal(x[0], want) and np.array_equal(x[1], want)
        assert np.array_equal(w, [0.5, 0.5])


def _dense_reference(x, g, m, w, lr, mu, peer, act):
    """Independent numpy fp64 statement: X_new = P (local step of X), P row-stochastic with
    P[j][j] = wh_j / W_j, P[j][i] = wh_i / W_j for every active i that chose j."""
    K = x.shape[0]
    act = act.astype(bool)
    x = x.astype(np.float64); g = g.astype(np.float64); m = m.astype(np.float64)
    m_new = np.where(act[:, None], mu * m + g, m)
    step_dir = m_new if mu != 0.0 else g
    y = np.where(act[:, None], x - lr * step_dir, x)
    wh = np.where(act, w / 2, w) if K >= 2 else w.copy()
    P = np.zeros((K, K))
    for j in range(K):
        P[j, j] = wh[j]
        for i in range(K):
            if act[i] and peer[i] == j:
                P[j, i] += wh[i]
    W = P.sum(axis=1)
    return (P / W[:, None]) @ y, m_new, W


@pytest.mark.parametrize("K,mu", [(2, 0.0), (3, 0.0), (3, 0.9), (4, 0.5)])
def test_bruteforce_every_schedule(K, mu):
    """I6: all (K-1)^K peer maps x all 2^K masks."""
    rng = np.random.default_rng(K * 10 + int(mu * 10))
    n, lr = 5, 0.125
    others = [[j for j in range(K) if j != i] for i in range(K)]
    checked = 0
    for peers in itertools.product(*others):
        for mask in itertools.product([0, 1], repeat=K):
            x = rng.normal(0, 1, (K, n)).astype(np.float32)
            g = rng.normal(0, 1, (K, n)).astype(np.float32)
            m = rng.normal(0, 1, (K, n)).astype(np.float32)
            w = rng.dirichlet(np.ones(K))
            act = np.array(mask, dtype=np.uint8)
            peer = np.where(act == 1, np.array(peers), -1).astype(np.int32)
            want_x, want_m, want_w = _dense_reference(x, g, m, w, lr, mu, peer, act)
            x2, m2, w2 = x.copy(), m.copy(), w.copy()
            oracle.layer_update(x2, g, m2, w2, lr, mu, 0, 0, 0, peer_in=peer, active_in=act)
            scale = np.abs(want_x).max()
            assert np.abs(x2 - want_x).max() <= 1e-6 * scale
            np.testing.assert_allclose(w2, want_w, rtol=1e-14)
            if mu != 0.0:
                assert np.abs(m2 - want_m).max() <= 1e-6 * np.abs(want_m).max()
            else:
                assert np.array_equal(m2, m)          # no momentum buffer is touched
            checked += 1
    assert checked == (K - 1) ** K * 2 ** K


def test_bruteforce_sampled_k5_and_drawn_schedule():
    """K = 5 on a random subset of schedules, plus schedules drawn by the oracle's own selector."""
    rng = np.random.default_rng(5)
    K, n = 5, 7
    for trial in range(400):
        act = rng.integers(0, 2, K).astype(np.uint8)
        peer = np.array([rng.choice([j for j in range(K) if j != i]) for i in range(K)], dtype=np.int32)
        peer = np.where(act == 1, peer, -1).astype(np.int32)
        x = rng.normal(0, 1, (K, n)).astype(np.float32)
        g = rng.normal(0, 1, (K, n)).astype(np.float32)
        m = rng.normal(0, 1, (K, n)).astype(np.float32)
        w = rng.dirichlet(np.ones(K))
        want_x, want_m, want_w = _dense_reference(x, g, m, w, 0.3, 0.9, peer, act)
        oracle.layer_update(x, g, m, w, 0.3, 0.9, 0, 0, 0, peer_in=peer, active_in=act)
        assert np.abs(x - want_x).max() <= 1e-6 * np.abs(want_x).max()
        np.testing.assert_allclose(w, want_w, rtol=1e-14)
    for step in range(50):
        K, L, seed, p = 8, 3, 11, 0.25
        peers, act = oracle.schedule(seed, step, L, K, 0, p)
        for layer in range(L):
            x = rng.normal(0, 1, (K, n)).astype(np.float32)
            g = rng.normal(0, 1, (K, n)).astype(np.float32)
            m = np.zeros_like(x)
            w = rng.dirichlet(np.ones(K))
            want_x, _, want_w = _dense_reference(x, g, m, w, 0.01, 0.0, peers[layer], act)
            oracle.layer_update(x, g, None, w, 0.01, 0.0, seed, step, layer, 0, p)
            assert np.abs(x - want_x).max() <= 1e-6 * np.abs(want_x).max()
            np.testing.assert_allclose(w, want_w, rtol=1e-14)


@pytest.mark.parametrize("K,p,mode", [(2, 0.0, 0), (4, 0.0, 0), (8, 0.25, 0), (16, 0.0, 1), (64, 0.25, 0)])
def test_mass_mean_convexity_consensus(K, p, mode):
    """I1, I2, I4, I5 over 150 pure-mix rounds (zero gradient)."""
    rng = np.random.default_rng(K)
    L, n, seed = 3, 33, 123
    o = oracle.Oracle([n] * L, K, lr=0.01, momentum=0.0, seed=seed, peer_mode=mode, skip_prob=p)
    for l in range(L):
        o.x[l][:] = rng.normal(0, 1, (K, n)).astype(np.float32)
    zeros = [np.zeros((K, n), dtype=np.float32) for _ in range(L)]
    wmean0 = [(o.w[l][:, None] * o.x[l].astype(np.float64)).sum(0) for l in range(L)]
    scale = max(np.abs(o.x[l]).max() for l in range(L))

    def wdist(l):
        xb = (o.w[l][:, None] * o.x[l].astype(np.float64)).sum(0)
        return float((o.w[l][:, None] * (o.x[l] - xb[None, :]) ** 2).sum())

    prev = [wdist(l) for l in range(L)]
    first = list(prev)
    wsum_t = np.zeros((L, K))
    for t in range(150):
        before = [x.copy() for x in o.x]
        peers, act = oracle.schedule(seed, t, L, K, mode, p)
        o.round(t, zeros)
        for l in range(L):
            assert abs(o.w[l].sum() - 1.0) <= 1e-15 * 8 and (o.w[l] > 0).all()              # I1
            wm = (o.w[l][:, None] * o.x[l].astype(np.float64)).sum(0)
            assert np.abs(wm - wmean0[l]).max() <= 4 * K * 2.0 ** -24 * scale * (1 + t / 50)  # I2
            d = wdist(l)
            assert d <= prev[l] * (1 + 1e-6) + 1e-12                                          # I4
            prev[l] = d
            for j in range(K):                                                                # I5
                grp = [before[l][j]] + [before[l][i] for i in range(K) if act[i] and peers[l][i] == j]
                lo, hi = np.min(grp, axis=0), np.max(grp, axis=0)
                tol = 2e-7 * np.maximum(np.abs(lo), np.abs(hi))
                assert (o.x[l][j] >= lo - tol).all() and (o.x[l][j] <= hi + tol).all()
                if len(grp) == 1:
                    assert np.array_equal(o.x[l][j], before[l][j])      # nobody pushed: untouched
        wsum_t += o.w
    for l in range(L):
        assert prev[l] < 1e-6 * first[l]                                                      # consensus reached
    if mode == 1:
        assert (o.w == o.w[0][None, :]).all()                                                 # I10
    # E[w_i] = 1/M: time-average of each weight near 1/K
    if K <= 16:
        assert np.abs(wsum_t / 150 - 1.0 / K).max() < 0.6 / K


@pytest.mark.parametrize("mu", [0.0, 0.9])
def test_k1_is_torch_sgd(mu):
    """I7: one worker => no peer, no mix; the path is torch.optim.SGD(momentum, dampening=0)."""
    torch.manual_seed(0)
    n, lr = 1000, 0.05
    p = torch.nn.Parameter(torch.randn(n))
    opt = torch.optim.SGD([p], lr=lr, momentum=mu)
    o = oracle.Oracle([n], 1, lr=lr, momentum=mu, seed=1)
    o.x[0][0] = p.detach().numpy()
    for t in range(12):
        g = torch.randn(n)
        p.grad = g.clone()
        opt.step()
        o.round(t, [g.numpy().reshape(1, n).copy()])
        # torch does not promise fused multiply-add: allow 1 ulp-scale difference per step
        np.testing.assert_allclose(o.x[0][0], p.detach().numpy(), rtol=0, atol=2e-7 * (t + 1) * 4)
        assert o.w[0, 0] == 1.0


@pytest.mark.parametrize("mu", [0.0, 0.9])
def test_consensus_fixed_point_follows_single_sgd(mu):
    """I8: identical replicas + identical gradients stay bit-identical and equal K=1 SGD."""
    rng = np.random.default_rng(2)
    K, n, lr = 8, 129, 0.01
    many = oracle.Oracle([n], K, lr=lr, momentum=mu, seed=4)
    one = oracle.Oracle([n], 1, lr=lr, momentum=mu, seed=4)
    x0 = rng.normal(0, 0.02, n).astype(np.float32)
    many.x[0][:] = x0[None, :]
    one.x[0][0] = x0
    for t in range(30):
        g = rng.normal(0, 1e-2, n).astype(np.float32)
        many.round(t, [np.repeat(g[None, :], K, 0).copy()])
        one.round(t, [g[None, :].copy()])
        assert (many.x[0] == many.x[0][0][None, :]).all()
        assert np.array_equal(many.x[0][0], one.x[0][0])


def test_layers_are_independent_of_order():
    """I9: forward-order, reverse-order and shuffled layer walks give identical bits."""
    rng = np.random.default_rng(3)
    K, numel, seed = 8, [40, 17, 96, 5], 21
    runs = []
    for order in ([3, 2, 1, 0], [0, 1, 2, 3], [2, 0, 3, 1]):
        o = oracle.Oracle(numel, K, lr=0.01, momentum=0.9, seed=seed, skip_prob=0.25)
        r = np.random.default_rng(99)
        for l, n in enumerate(numel):
            o.x[l][:] = r.normal(0, 0.02, (K, n)).astype(np.float32)
        for t in range(10):
            gs = [r.normal(0, 1e-2, (K, n)).astype(np.float32) for n in numel]
            for l in order:
                o.layer_update(t, l, gs[l])
        runs.append(o)
    for o in runs[1:]:
        for l in range(len(numel)):
            assert np.array_equal(o.x[l], runs[0].x[l]) and np.array_equal(o.m[l], runs[0].m[l])
        assert np.array_equal(o.w, runs[0].w)


def test_straggler_semantics():
    """PAPER.md:229 'the straggler keeps receiving updates' + R10: an inactive replica's x
    changes iff somebody pushed to it, its momentum never changes, its weight is not halved."""
    rng = np.random.default_rng(8)
    K, n, seed, p = 8, 50, 3, 0.25
    o = oracle.Oracle([n], K, lr=0.01, momentum=0.9, seed=seed, skip_prob=p)
    o.x[0][:] = rng.normal(0, 0.02, (K, n)).astype(np.float32)
    seen_inactive_recv = seen_inactive_idle = 0
    for t in range(60):
        peers, act = oracle.schedule(seed, t, 1, K, 0, p)
        xb, mb, wb = o.x[0].copy(), o.m[0].copy(), o.w[0].copy()
        o.round(t, [rng.normal(0, 1e-2, (K, n)).astype(np.float32)])
        for i in range(K):
            if act[i]:
                continue
            recv = sum(wb[s] / 2 for s in range(K) if act[s] and peers[0][s] == i)
            assert np.array_equal(o.m[0][i], mb[i])
            assert o.w[0][i] == pytest.approx(wb[i] + recv, rel=1e-15)
            if recv == 0:
                assert np.array_equal(o.x[0][i], xb[i]); seen_inactive_idle += 1
            else:
                assert not np.array_equal(o.x[0][i], xb[i]); seen_inactive_recv += 1
    assert seen_inactive_recv > 0 and seen_inactive_idle > 0


def test_fp32_tracks_fp64_shadow_100_rounds():
    """north_star: fp32 within 1e-5 (scale-relative, R15) of exact arithmetic after 100 rounds."""
    rng = np.random.default_rng(13)
    K, numel, seed = 8, [300, 41], 17
    o32 = oracle.Oracle(numel, K, lr=3e-4, momentum=0.9, seed=seed, skip_prob=0.1)
    o64 = oracle.Oracle(numel, K, lr=3e-4, momentum=0.9, seed=seed, skip_prob=0.1, f64=True)
    for l, n in enumerate(numel):
        x0 = rng.normal(0, 0.02, (K, n)).astype(np.float32)
        o32.x[l][:] = x0
        o64.x[l][:] = x0
    for t in range(100):
        gs = [rng.normal(0, 1e-3, (K, n)).astype(np.float32) for n in numel]
        o32.round(t, gs)
        o64.round(t, gs)
        assert np.array_equal(o32.w, o64.w)
    for l in range(len(numel)):
        err = np.abs(o32.x[l] - o64.x[l]).max() / np.abs(o64.x[l]).max()
        assert err <= 1e-5, err
