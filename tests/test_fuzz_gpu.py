"""Seeded random configurations of the whole rule against the oracle (GPU).  compute-sanitizer is
closed on this pool, so breadth stands in for it: random replica counts (odd, even, around the TMA
box limits), ragged layer sizes on both sides of tile boundaries, every optimiser x mixer, both peer
modes, random and delay-mode stragglers, launches small enough for the single-launch path and large
enough for the two-launch path with 2-D tile loads, per-layer events mixed with whole rounds."""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import REL_TOL_ROUND, max_ulp, rel_err
from paper_2410_05985_b200 import (MIX_LOSSY, MIX_PUSHSUM, MIX_SYMMETRIC, OPT_ADAMW, OPT_SGD, WHAT_G, WHAT_M, WHAT_V,
                                   WHAT_X, LayUp)

pytestmark = pytest.mark.gpu


def _draw(seed):
    r = np.random.default_rng(seed)
    K = int(r.choice([1, 2, 3, 4, 5, 7, 8, 9, 15, 16, 17, 31, 32, 33, 48, 63, 64, 65, 100, 128, 255, 256, 257, 300]))
    big = seed % 5 == 0 and K <= 64                      # every fifth case: more than 4 waves of work items
    L = int(r.integers(1, 6))
    if big:
        per_tile = max(8, 1024 // K) * 4
        numel = [int(per_tile * r.integers(700, 1200) + r.integers(0, per_tile)) for _ in range(L)]
        numel[0] = int(3000 * per_tile + r.integers(1, 100))
    else:
        numel = [int(r.choice([1, 3, 31, 32, 33, 100, 255, 256, 257, 1000, 4095, 4097, 20000])) + int(r.integers(0, 50))
                 for _ in range(L)]
    opt = int(r.choice([OPT_SGD, OPT_SGD, OPT_ADAMW]))
    cfg = dict(K=K, numel=numel, lr=float(r.choice([1e-3, 0.01, 0.3])), momentum=float(r.choice([0.0, 0.9])) if opt == OPT_SGD else 0.0,
               seed=int(r.integers(0, 2**40)), peer_mode=int(r.integers(0, 2)), skip_prob=float(r.choice([0.0, 0.0, 0.25, 0.6])),
               delay_replica=int(r.integers(0, K)), delay_rounds=int(r.choice([0, 0, 0, 2])), optimizer=opt,
               mix_mode=int(r.choice([MIX_PUSHSUM, MIX_PUSHSUM, MIX_LOSSY, MIX_SYMMETRIC])),
               weight_decay=float(r.choice([0.0, 0.01])), beta1=0.9, beta2=float(r.choice([0.95, 0.999])), eps=1e-8)
    return cfg, big


@pytest.mark.parametrize("case", range(100))
def test_random_configuration_matches_the_oracle(case):
    cfg, big = _draw(1000 + case)
    K, numel = cfg["K"], cfg["numel"]
    kw = {k: cfg[k] for k in ("delay_replica", "delay_rounds", "optimizer", "mix_mode", "weight_decay", "beta1", "beta2", "eps")}
    lu = LayUp(K, numel, cfg["lr"], cfg["momentum"], cfg["seed"], cfg["peer_mode"], cfg["skip_prob"], **kw)
    ref = oracle.Oracle(numel, K, cfg["lr"], cfg["momentum"], cfg["seed"], cfg["peer_mode"], cfg["skip_prob"], **kw)
    gen = torch.Generator(device="cuda").manual_seed(case)
    L = len(numel)
    for l in range(L):
        lu.view(WHAT_X, l).normal_(0, 0.02, generator=gen)
        ref.x[l][:] = lu.view(WHAT_X, l).cpu().numpy()
    rounds = 2 if big else 5
    for step in range(rounds):
        grads = []
        for l in range(L):
            lu.view(WHAT_G, l).normal_(0, 1e-2, generator=gen)
            grads.append(lu.view(WHAT_G, l).cpu().numpy())
        peer, active = lu.layup_schedule(step)
        rp, ra = oracle.schedule(cfg["seed"], step, L, K, cfg["peer_mode"], cfg["skip_prob"], cfg["delay_replica"], cfg["delay_rounds"])
        assert np.array_equal(peer, rp) and np.array_equal(active, ra), cfg
        if step % 2 == 0:
            lu.layup_round(step)
        else:
            for l in reversed(range(L)):
                lu.layup_layer_update(step, l)
        lu.layup_sync()
        ref.round(step, grads)
        for l in range(L):
            pairs = [(WHAT_X, ref.x[l])] + ([(WHAT_M, ref.m[l])] if ref.m is not None else []) + \
                    ([(WHAT_V, ref.v[l])] if ref.v is not None else [])
            for what, want in pairs:
                got = lu.view(what, l).cpu().numpy()
                assert rel_err(got, want) <= REL_TOL_ROUND, (cfg, step, l, what)
                assert max_ulp(got, want) == 0, (cfg, step, l, what)
        assert np.array_equal(lu.layup_weights(), ref.w), (cfg, step)
    lu.close()
