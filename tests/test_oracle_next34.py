"""Pins for the widened rule (CPU only): SURVEY.md 8(f) NEXT-3 (AdamW, coupled weight decay)
and NEXT-4 (contention-lossy and symmetric mixers).  As in test_oracle_pins.py nothing here
re-types the oracle's formula: worked examples derived by hand (tests/golden/W4-W6), the
library optimisers torch.optim.{AdamW, Adam, SGD} for K = 1, dense matrix products written
independently in numpy fp64 over EVERY schedule of tiny problems, and invariants."""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

import oracle
from oracle import MIX_LOSSY, MIX_PUSHSUM, MIX_SYMMETRIC, OPT_ADAMW, OPT_SGD

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _read_rounds(name):
    """-> (header dict, [per-round dict]); a 'round' line starts a new block."""
    head, rounds, cur = {}, [], None
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, *v = line.split()
            if k == "round":
                cur = {}
                rounds.append(cur)
                continue
            (head if cur is None or k in ("K", "lr", "wd", "beta1", "beta2", "eps") else cur)[k] = \
                [float(Fraction(t)) for t in v]
    return head, rounds


def test_w4_adamw_two_steps_then_push():
    head, rounds = _read_rounds("W4_adamw_two_steps.txt")
    K = int(head["K"][0])
    r0 = rounds[0]
    for dt in (np.float32, np.float64):
        x = np.array(r0["x_before"], dtype=dt).reshape(K, 1)
        m = np.array(r0["m_before"], dtype=dt).reshape(K, 1)
        v = np.array(r0["v_before"], dtype=dt).reshape(K, 1)
        g = np.array(r0["g"], dtype=np.float32).reshape(K, 1)
        w = np.array(r0["w_before"], dtype=np.float64)
        bpow, tc = np.ones((K, 2)), np.zeros(K, dtype=np.int64)
        peer = np.array(r0["peer"], dtype=np.int32)
        act = np.array(r0["active"], dtype=np.uint8)
        for r in rounds:
            oracle.layer_update_ex(x, g, m, v, w, bpow, tc, lr=head["lr"][0], wd=head["wd"][0],
                                   beta1=head["beta1"][0], beta2=head["beta2"][0], eps=head["eps"][0],
                                   optimizer=OPT_ADAMW, peer_in=peer, active_in=act)
            tol = 3e-7 if dt == np.float32 else 2e-8     # lr = 0.1 is itself rounded to fp32 on both paths
            np.testing.assert_allclose(x[:, 0], r["x_after"], rtol=tol)
            np.testing.assert_allclose(m[:, 0], r["m_after"], rtol=1e-7)
            np.testing.assert_allclose(v[:, 0], r["v_after"], rtol=1e-7)
            np.testing.assert_allclose(w, r["w_after"], rtol=1e-15)
        assert list(tc) == [2, 0]


@pytest.mark.parametrize("name", ["W5_contention_last_writer.txt", "W6_symmetric_pairwise.txt"])
def test_w5_w6_mixers(name):
    head, _ = _read_rounds(name)
    K, mode = int(head["K"][0]), int(head["mix_mode"][0])
    for dt in (np.float32, np.float64):
        x = np.array(head["x_before"], dtype=dt).reshape(K, 1)
        g = np.zeros((K, 1), dtype=np.float32)
        w = np.array(head["w_before"], dtype=np.float64)
        oracle.layer_update_ex(x, g, None, None, w, None, None, lr=0.5, mix_mode=mode,
                               peer_in=np.array(head["peer"], dtype=np.int32), active_in=np.ones(K, dtype=np.uint8))
        np.testing.assert_allclose(x[:, 0], head["x_after"], rtol=1e-7)
        np.testing.assert_allclose(w, head["w_after"], rtol=1e-15)


# ---- library reductions: one worker => the path is the library optimiser --------------------
@pytest.mark.parametrize("wd,amsgrad_free_adam", [(0.0, True), (0.0031235, False), (0.1, False)])
def test_k1_is_torch_adamw(wd, amsgrad_free_adam):
    """K = 1: no peer, no mix; AdamW with PyTorch's convention (bias correction, decoupled decay).
    wd = 0.0031235 and lr = 7.5249e-4 are the paper's GPT-2 medium values."""
    torch.manual_seed(1)
    n, lr, b1, b2, eps = 2000, 7.5249e-4, 0.9, 0.95, 1e-8
    p = torch.nn.Parameter(torch.randn(n) * 0.02)
    if amsgrad_free_adam:
        opt = torch.optim.Adam([p], lr=lr, betas=(b1, b2), eps=eps)          # Adam == AdamW with wd = 0
    else:
        opt = torch.optim.AdamW([p], lr=lr, betas=(b1, b2), eps=eps, weight_decay=wd)
    o = oracle.Oracle([n], 1, lr=lr, seed=1, optimizer=OPT_ADAMW, weight_decay=wd, beta1=b1, beta2=b2, eps=eps)
    sh = oracle.Oracle([n], 1, lr=lr, seed=1, optimizer=OPT_ADAMW, weight_decay=wd, beta1=b1, beta2=b2, eps=eps, f64=True)
    o.x[0][0] = p.detach().numpy()
    sh.x[0][0] = p.detach().numpy()
    for t in range(40):
        g = torch.randn(n) * 1e-3
        if t % 7 == 3:
            g[::5] *= 100.0                                                   # heavy tail as configs[2]
        p.grad = g.clone()
        opt.step()
        gn = g.numpy().reshape(1, n).copy()
        o.round(t, [gn])
        sh.round(t, [gn])
        ref = p.detach().numpy()
        scale = np.abs(ref).max()
        assert np.abs(o.x[0][0] - ref).max() <= 2e-7 * (t + 1) * scale
        assert np.abs(sh.x[0][0] - ref).max() <= 2e-7 * (t + 1) * scale
        st = opt.state[p]
        np.testing.assert_allclose(o.m[0][0], st["exp_avg"].numpy(), rtol=0, atol=1e-6 * np.abs(st["exp_avg"].numpy()).max())
        np.testing.assert_allclose(o.v[0][0], st["exp_avg_sq"].numpy(), rtol=0, atol=1e-6 * np.abs(st["exp_avg_sq"].numpy()).max())
    assert o.tcount[0, 0] == 40 and o.w[0, 0] == 1.0


@pytest.mark.parametrize("mu,wd", [(0.0, 0.005), (0.9, 0.0001), (0.9, 0.014)])
def test_k1_is_torch_sgd_with_weight_decay(mu, wd):
    """Coupled decay d = g + wd*x (torch.optim.SGD weight_decay); wd values from PAPER.md:416-443."""
    torch.manual_seed(2)
    n, lr = 1500, 0.035
    p = torch.nn.Parameter(torch.randn(n))
    opt = torch.optim.SGD([p], lr=lr, momentum=mu, weight_decay=wd)
    o = oracle.Oracle([n], 1, lr=lr, momentum=mu, seed=1, weight_decay=wd)
    o.x[0][0] = p.detach().numpy()
    for t in range(15):
        g = torch.randn(n)
        p.grad = g.clone()
        opt.step()
        o.round(t, [g.numpy().reshape(1, n).copy()])
        np.testing.assert_allclose(o.x[0][0], p.detach().numpy(), rtol=0, atol=2e-7 * (t + 1) * 4)
    # and the decay term is really there: against the undecayed run the iterates differ
    o2 = oracle.Oracle([n], 1, lr=lr, momentum=mu, seed=1)
    assert o2.wd == 0.0


def test_adamw_first_step_is_sign_descent():
    """Closed form: from m = v = 0 the first AdamW step is x(1-lr*wd) - lr*g/(|g|+eps)."""
    rng = np.random.default_rng(3)
    K, n, lr, wd, eps = 3, 64, 0.01, 0.25, 1e-8
    x = rng.normal(0, 1, (K, n)).astype(np.float32)
    g = rng.normal(0, 1, (K, n)).astype(np.float32)
    want = x.astype(np.float64) * (1 - np.float32(lr).astype(np.float64) * wd) - np.float64(np.float32(lr)) * g / (np.abs(g) + eps)
    m, v = np.zeros_like(x), np.zeros_like(x)
    w = np.full(K, 1 / 3)
    bpow, tc = np.ones((K, 2)), np.zeros(K, dtype=np.int64)
    # every worker pushes to an inactive-free ring but we look at y through a mask with no push: all idle peers
    act = np.array([1, 0, 0], dtype=np.uint8)
    peer = np.array([1, -1, -1], dtype=np.int32)
    x2 = x.copy()
    oracle.layer_update_ex(x2, g, m, v, w, bpow, tc, lr=lr, wd=wd, beta1=0.9, beta2=0.999, eps=eps,
                           optimizer=OPT_ADAMW, peer_in=peer, active_in=act)
    np.testing.assert_allclose(x2[0], want[0], rtol=0, atol=3e-7 * np.abs(want[0]).max())
    assert np.array_equal(x2[2], x[2])                       # idle, not a receiver: untouched
    assert (m[1:] == 0).all() and (v[1:] == 0).all() and list(tc) == [1, 0, 0]
    assert np.array_equal(bpow[1:], np.ones((2, 2)))         # a straggler's optimiser state does not move


# ---- dense references over every schedule ------------------------------------------------------
def _local_sgd64(x, g, act, lr):
    return np.where(act.astype(bool)[:, None], x.astype(np.float64) - lr * g.astype(np.float64), x.astype(np.float64))


def _dense_lossy(y, w, peer, act):
    """X_new = P y with only the highest-index sender of each receiver in P; the weight of every
    other colliding sender is halved away and never arrives."""
    K = y.shape[0]
    wh = np.where(act.astype(bool), w / 2, w)
    P = np.zeros((K, K))
    for j in range(K):
        P[j, j] = wh[j]
        senders = [i for i in range(K) if act[i] and peer[i] == j]
        if senders:
            P[j, max(senders)] += wh[max(senders)]
    W = P.sum(axis=1)
    return (P / W[:, None]) @ y, W


def _dense_symmetric(y, peer, act):
    """Product of pairwise-averaging matrices A_i = I - (e_i - e_j)(e_i - e_j)^T / 2, i ascending."""
    K = y.shape[0]
    T = np.eye(K)
    for i in range(K):
        if act[i] and peer[i] >= 0:
            d = np.zeros(K); d[i] = 1.0; d[peer[i]] -= 1.0
            T = (np.eye(K) - np.outer(d, d) / 2.0) @ T
    return T @ y, T


@pytest.mark.parametrize("K", [2, 3, 4])
@pytest.mark.parametrize("mode", [MIX_LOSSY, MIX_SYMMETRIC])
def test_bruteforce_every_schedule_variant_mixers(K, mode):
    rng = np.random.default_rng(100 * K + mode)
    n, lr = 5, 0.125
    others = [[j for j in range(K) if j != i] for i in range(K)]
    checked = 0
    for peers in itertools.product(*others):
        for mask in itertools.product([0, 1], repeat=K):
            x = rng.normal(0, 1, (K, n)).astype(np.float32)
            g = rng.normal(0, 1, (K, n)).astype(np.float32)
            w = rng.dirichlet(np.ones(K))
            act = np.array(mask, dtype=np.uint8)
            peer = np.where(act == 1, np.array(peers), -1).astype(np.int32)
            y = _local_sgd64(x, g, act, lr)
            if mode == MIX_LOSSY:
                want_x, want_w = _dense_lossy(y, w, peer, act)
            else:
                want_x, T = _dense_symmetric(y, peer, act)
                want_w = w.copy()
                np.testing.assert_allclose(T.sum(axis=0), 1.0, atol=1e-15)   # doubly stochastic
                np.testing.assert_allclose(T.sum(axis=1), 1.0, atol=1e-15)
            for dt in (np.float32, np.float64):
                x2, w2 = x.astype(dt), w.copy()
                oracle.layer_update_ex(x2, g, None, None, w2, None, None, lr=lr, mix_mode=mode,
                                       peer_in=peer, active_in=act)
                tol = 1e-6 if dt == np.float32 else 1e-12
                assert np.abs(x2 - want_x).max() <= tol * np.abs(want_x).max()
                np.testing.assert_allclose(w2, want_w, rtol=1e-14)
            checked += 1
    assert checked == (K - 1) ** K * 2 ** K


def test_lossy_equals_lossless_without_collisions_and_loses_mass_with():
    rng = np.random.default_rng(7)
    K, n = 8, 33
    for trial in range(200):
        x = rng.normal(0, 1, (K, n)).astype(np.float32)
        g = rng.normal(0, 1, (K, n)).astype(np.float32)
        w = rng.dirichlet(np.ones(K))
        if trial % 2 == 0:                                   # a derangement: nobody collides
            while True:
                perm = rng.permutation(K)
                if (perm != np.arange(K)).all():
                    break
            peer = perm.astype(np.int32)
        else:
            peer = np.array([rng.choice([j for j in range(K) if j != i]) for i in range(K)], dtype=np.int32)
        act = np.ones(K, dtype=np.uint8)
        xa, wa, xb, wb = x.copy(), w.copy(), x.copy(), w.copy()
        oracle.layer_update_ex(xa, g, None, None, wa, None, None, lr=0.1, mix_mode=MIX_PUSHSUM, peer_in=peer, active_in=act)
        oracle.layer_update_ex(xb, g, None, None, wb, None, None, lr=0.1, mix_mode=MIX_LOSSY, peer_in=peer, active_in=act)
        counts = np.bincount(peer, minlength=K)
        if (counts <= 1).all():
            assert np.array_equal(xa, xb) and np.array_equal(wa, wb)
        else:
            lost = sum(w[i] / 2 for j in range(K) for i in np.nonzero(peer == j)[0][:-1])
            np.testing.assert_allclose(wb.sum(), w.sum() - lost, rtol=1e-14)
            assert wb.sum() < wa.sum()
        np.testing.assert_allclose(wa.sum(), w.sum(), rtol=1e-14)
        # convexity of whatever landed (PAPER.md:101 coefficients sum to one)
        y = x - np.float32(0.1) * g
        lo, hi = y.min(axis=0), y.max(axis=0)
        assert (xb >= lo - 1e-6).all() and (xb <= hi + 1e-6).all()


@pytest.mark.parametrize("K,p", [(2, 0.0), (8, 0.0), (16, 0.25), (64, 0.0)])
def test_symmetric_conserves_plain_mean_and_contracts(K, p):
    """Doubly-stochastic mixing: the plain replica mean of a pure mix is conserved and the
    unweighted disagreement sum_i ||x_i - xbar||^2 never grows (each exchange is a projection)."""
    rng = np.random.default_rng(K)
    n = 40
    o = oracle.Oracle([n], K, lr=0.0, seed=9, skip_prob=p, mix_mode=MIX_SYMMETRIC)
    o.x[0][:] = rng.normal(0, 1, (K, n)).astype(np.float32)
    mean0 = o.x[0].astype(np.float64).mean(axis=0)
    prev = o.disagreement()[0].sum()
    first = prev
    for t in range(60):
        o.round(t, [np.zeros((K, n), dtype=np.float32)])
        d = o.disagreement()[0].sum()
        assert d <= prev * (1 + 1e-6) + 1e-12
        prev = d
        np.testing.assert_allclose(o.x[0].astype(np.float64).mean(axis=0), mean0, atol=4 * K * 2**-24 * (t + 1))
        assert np.array_equal(o.w[0], np.full(K, 1.0 / K))
    assert prev < 1e-3 * first
    if K == 2 and p == 0.0:
        assert np.array_equal(o.x[0][0], o.x[0][1])


def test_k2_symmetric_is_exact_average():
    rng = np.random.default_rng(0)
    x = (rng.integers(-2**16, 2**16, size=(2, 257)) / 1024.0).astype(np.float32)
    want = ((x[0].astype(np.float64) + x[1]) / 2).astype(np.float32)
    w = np.array([0.5, 0.5])
    oracle.layer_update_ex(x, np.zeros_like(x), None, None, w, None, None, lr=0.1, mix_mode=MIX_SYMMETRIC, seed=5, step=3)
    assert np.array_equal(x[0], want) and np.array_equal(x[1], want)


@pytest.mark.parametrize("mode", [MIX_PUSHSUM, MIX_LOSSY, MIX_SYMMETRIC])
def test_adamw_consensus_fixed_point_and_straggler_state(mode):
    """Identical replicas + identical gradients stay bit-identical and follow K = 1 AdamW under every
    mixer; with stragglers a worker's (m, v, t) move only in the rounds it is active."""
    rng = np.random.default_rng(11)
    K, n = 6, 65
    kw = dict(lr=1e-3, seed=4, optimizer=OPT_ADAMW, weight_decay=0.01, beta1=0.9, beta2=0.95, eps=1e-8)
    many = oracle.Oracle([n], K, mix_mode=mode, **kw)
    one = oracle.Oracle([n], 1, **kw)
    x0 = rng.normal(0, 0.02, n).astype(np.float32)
    many.x[0][:] = x0[None, :]
    one.x[0][0] = x0
    for t in range(25):
        g = rng.normal(0, 1e-2, n).astype(np.float32)
        many.round(t, [np.repeat(g[None, :], K, 0).copy()])
        one.round(t, [g[None, :].copy()])
        assert (many.x[0] == many.x[0][0][None, :]).all()
        assert np.array_equal(many.x[0][0], one.x[0][0])
    lag = oracle.Oracle([n], K, mix_mode=mode, skip_prob=0.4, **kw)
    lag.x[0][:] = rng.normal(0, 0.02, (K, n)).astype(np.float32)
    for t in range(25):
        _, act = oracle.schedule(4, t, 1, K, 0, 0.4)
        m0, v0, t0, b0 = lag.m[0].copy(), lag.v[0].copy(), lag.tcount[0].copy(), lag.bpow[0].copy()
        lag.round(t, [rng.normal(0, 1e-2, (K, n)).astype(np.float32)])
        for i in range(K):
            if act[i]:
                assert lag.tcount[0, i] == t0[i] + 1 and not np.array_equal(lag.m[0][i], m0[i])
            else:
                assert lag.tcount[0, i] == t0[i] and np.array_equal(lag.m[0][i], m0[i])
                assert np.array_equal(lag.v[0][i], v0[i]) and np.array_equal(lag.bpow[0][i], b0[i])
    np.testing.assert_allclose(lag.bpow[0][:, 0], np.float64(np.float32(0.9)) ** lag.tcount[0], rtol=1e-13)


@pytest.mark.parametrize("opt,mode", [(OPT_ADAMW, MIX_PUSHSUM), (OPT_SGD, MIX_LOSSY), (OPT_SGD, MIX_SYMMETRIC),
                                      (OPT_ADAMW, MIX_SYMMETRIC)])
def test_fp32_tracks_fp64_shadow_100_rounds_widened(opt, mode):
    rng = np.random.default_rng(21)
    K, numel = 8, [300, 77]
    kw = dict(lr=3e-4, momentum=0.9 if opt == OPT_SGD else 0.0, seed=5, skip_prob=0.1, optimizer=opt, mix_mode=mode,
              weight_decay=0.01, beta1=0.9, beta2=0.95, eps=1e-8)
    a = oracle.Oracle(numel, K, **kw)
    b = oracle.Oracle(numel, K, f64=True, **kw)
    for l, n in enumerate(numel):
        x0 = rng.normal(0, 0.02, (K, n)).astype(np.float32)
        a.x[l][:] = x0
        b.x[l][:] = x0
    for t in range(100):
        gs = [rng.normal(0, 1e-3, (K, n)).astype(np.float32) for n in numel]
        a.round(t, gs)
        b.round(t, gs)
    for l in range(len(numel)):
        err = np.abs(a.x[l] - b.x[l]).max() / np.abs(b.x[l]).max()
        assert err <= 1e-5, (l, err)
        np.testing.assert_allclose(a.w[l], b.w[l], rtol=1e-13)
