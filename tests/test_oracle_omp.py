"""Pins of the two oracle additions of round 2 (pytest -m "not gpu"):

* oracle_mix_tables -- the scalar half of the Peer Update (sender lists, alpha = w_i/(w_i+w_j),
  PAPER.md:101) stated on its own so that the tables the CUDA path consumed can be compared with
  it.  Pinned against the hand-derived coefficients of worked example W1 (tests/golden/), against
  an independent exact-rational restatement of PAPER.md:101 on every schedule of K <= 4, and
  against oracle_layer_update_ex itself (applying the listed pushes reproduces its result).
* the -fopenmp build of the SAME source (bench.py's all-cores baseline) is bit-identical to the
  serial build for every optimiser and mixer."""
import itertools
from fractions import Fraction

import numpy as np
import pytest

import oracle
from oracle import MIX_LOSSY, MIX_PUSHSUM, MIX_SYMMETRIC, OPT_ADAMW, OPT_SGD


def test_mix_tables_worked_example_w1():
    # tests/golden/W1_three_workers.txt: peers 0->1, 1->2, 2->1; "from 0: a=1/2", "from 2: a=1/3", "from 1: a=1/2"
    off, snd, al, w = oracle.mix_tables([1 / 3] * 3, [1, 2, 1], [1, 1, 1])
    assert off.tolist() == [0, 0, 2, 3] and snd.tolist() == [0, 2, 1]
    assert al.tolist() == [np.float32(0.5), np.float32(1 / 3), np.float32(0.5)]
    assert w.tolist() == [1 / 6, 0.5, 1 / 3]


def _exact_tables(w, peer, act, lossy):
    """PAPER.md:101 in exact rationals: halve every sender, then per receiver fold the senders in
    ascending index: alpha = w_i/(w_i+w_j), w_j += w_i."""
    K = len(w)
    wh = [Fraction(w[i]) / 2 if act[i] else Fraction(w[i]) for i in range(K)]
    rows, w_new = [], []
    for j in range(K):
        W = wh[j]
        snd = [i for i in range(K) if act[i] and peer[i] == j]
        if lossy and snd:
            snd = snd[-1:]
        row = []
        for i in snd:
            row.append((i, wh[i] / (W + wh[i])))
            W += wh[i]
        rows.append(row)
        w_new.append(W)
    return rows, w_new


@pytest.mark.parametrize("K", [2, 3, 4])
@pytest.mark.parametrize("mode", [MIX_PUSHSUM, MIX_LOSSY])
def test_mix_tables_every_schedule_against_exact_rationals(K, mode):
    rng = np.random.default_rng(K)
    others = [[j for j in range(K) if j != i] for i in range(K)]
    for peer in itertools.product(*others):
        for mask in itertools.product([0, 1], repeat=K):
            # dyadic weights (what push-sum produces) so that the rationals are exact in fp64
            w = (rng.integers(1, 64, K) / 256.0).astype(np.float64)
            pr = [p if a else -1 for p, a in zip(peer, mask)]
            off, snd, al, w_new = oracle.mix_tables(w, pr, mask, mode)
            rows, w_want = _exact_tables(w.tolist(), pr, mask, mode == MIX_LOSSY)
            for j in range(K):
                got = list(zip(snd[off[j]:off[j + 1]].tolist(), al[off[j]:off[j + 1]].tolist()))
                assert [g[0] for g in got] == [r[0] for r in rows[j]]
                for (_, a), (_, want) in zip(got, rows[j]):
                    assert a == np.float32(float(want))          # fp64 quotient of dyadics, rounded once
                assert w_new[j] == float(w_want[j])


@pytest.mark.parametrize("mode", [MIX_PUSHSUM, MIX_LOSSY])
def test_mix_tables_reproduce_the_layer_update(mode):
    """Applying the listed pushes one by one (x_j <- x_j + alpha (y_i - x_j), fp32) gives what
    oracle_layer_update_ex computes, and the weights agree bit for bit."""
    rng = np.random.default_rng(5)
    for K in (5, 8, 33):
        n = 64
        w = np.full(K, 1.0 / K)
        x = rng.standard_normal((K, n)).astype(np.float32)
        for step in range(6):
            g = np.zeros((K, n), dtype=np.float32)
            peer, act = oracle.schedule(11, step, 1, K, 0, 0.25)
            off, snd, al, w_new = oracle.mix_tables(w, peer[0], act, mode)
            want = x.copy()
            for j in range(K):
                acc = x[j].copy()
                for k in range(off[j], off[j + 1]):
                    d = x[snd[k]] - acc
                    acc = (acc.astype(np.float64) + np.float64(al[k]) * d.astype(np.float64)).astype(np.float32)
                want[j] = acc
            oracle.layer_update_ex(x, g, None, None, w, None, None, lr=0.0, mix_mode=mode, seed=11, step=step, layer=0,
                                   skip_prob=0.25)
            assert np.array_equal(w, w_new)
            assert np.abs(x - want).max() <= 2.0 ** -22 * np.abs(want).max()   # fmaf vs double-rounded emulation
    off, snd, al, w_new = oracle.mix_tables([0.25] * 4, [1, 0, 3, 2], [1, 1, 1, 1], MIX_SYMMETRIC)
    assert off.tolist() == [0] * 5 and snd.size == 0 and w_new.tolist() == [0.25] * 4


@pytest.mark.parametrize("opt,mix,mu,wd", [(OPT_SGD, MIX_PUSHSUM, 0.0, 0.0), (OPT_SGD, MIX_PUSHSUM, 0.9, 0.01),
                                           (OPT_SGD, MIX_LOSSY, 0.9, 0.0), (OPT_SGD, MIX_SYMMETRIC, 0.0, 0.0),
                                           (OPT_ADAMW, MIX_PUSHSUM, 0.0, 0.01), (OPT_ADAMW, MIX_SYMMETRIC, 0.0, 0.0)])
def test_openmp_build_is_bit_identical(opt, mix, mu, wd):
    K, numel = 6, [70001, 33, 40000]                      # above and below the parallel threshold
    rng = np.random.default_rng(3)
    x0 = [rng.standard_normal((K, n)).astype(np.float32) * 0.02 for n in numel]
    grads = [[rng.standard_normal((K, n)).astype(np.float32) * 1e-2 for n in numel] for _ in range(4)]
    outs = []
    try:
        for omp in (False, True):
            oracle.use_omp(omp)
            ref = oracle.Oracle(numel, K, 1e-2, mu, 9, 0, 0.25, optimizer=opt, mix_mode=mix, weight_decay=wd)
            for l in range(len(numel)):
                ref.x[l][:] = x0[l]
            for step in range(4):
                ref.round(step, grads[step])
            outs.append([a.copy() for a in ref.x] + ([a.copy() for a in ref.m] if ref.m else []) + [ref.w.copy()])
    finally:
        oracle.use_omp(False)
    for a, b in zip(*outs):
        assert np.array_equal(a, b)
