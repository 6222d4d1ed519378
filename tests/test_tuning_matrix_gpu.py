"""Every field of layup_tuning (include/layup.h) selects WHICH kernel runs and must not change a
single result bit: each block below runs the whole rule -- SGD, momentum and AdamW, the three
mixers, all-active and straggler rounds, whole rounds and per-layer events, ragged layers -- and is
compared with the oracle bit for bit (Alg. 1; mask PAPER.md:220-229)."""
import numpy as np
import pytest
import torch

import oracle
from _util import max_ulp
from paper_2410_05985_b200 import (LAYUP_EINVAL, MIX_LOSSY, MIX_PUSHSUM, MIX_SYMMETRIC, OPT_ADAMW, OPT_SGD, WHAT_G, WHAT_M, WHAT_V,
                                   WHAT_X, LayUp, LayUpError)

pytestmark = pytest.mark.gpu

# the persistent blocks carry fused = 2 (never): these layers are small enough for the single-launch
# path, which would otherwise run instead of the ring kernel at K <= 16
BLOCKS = [dict(), dict(launch_shape=2, fused=2), dict(launch_shape=2, stages=2, fused=2), dict(launch_shape=2), dict(engine=2),
          dict(tma2d=1), dict(tma2d=2),
          dict(variant=4), dict(variant=5), dict(variant=6), dict(variant=7), dict(pdl=2), dict(fused=2),
          dict(fused_waves=64), dict(tile_items=256), dict(tile_items=4096),
          dict(launch_shape=2, variant=1, group_threads=512, fused=2)]
# only a forced thread shape or tile size may be refused at init (a shape that cannot hold the tile of
# this K / optimiser says LAYUP_EINVAL); every other block must come up for every case
MAY_REFUSE = ("variant", "tile_items")


def _case(K, case):
    r = np.random.default_rng(case * 100 + K)
    numel = [int(256 * r.integers(100, 300) + r.integers(0, 256)) for _ in range(3)] + [int(r.integers(1, 300))]
    opt = [OPT_SGD, OPT_SGD, OPT_ADAMW][case % 3]
    mom = 0.9 if case % 3 == 1 else 0.0
    skip = [0.0, 0.25, 0.6][(case // 3 + case) % 3]
    mix = [MIX_PUSHSUM, MIX_LOSSY, MIX_SYMMETRIC, MIX_PUSHSUM][case % 4]
    kw = dict(optimizer=opt, mix_mode=mix, weight_decay=0.01 if case % 2 else 0.0, beta1=0.9, beta2=0.999, eps=1e-8)
    return numel, mom, skip, kw


@pytest.mark.parametrize("K", [5, 16, 64])
@pytest.mark.parametrize("block", BLOCKS, ids=lambda b: ",".join("%s=%d" % kv for kv in b.items()) or "defaults")
def test_tuning_block_changes_no_bit(block, K):
    ran = 0
    for case in (0, 1, 2, 4):         # SGD, momentum, AdamW x mixers x skip 0 / 0.25 / 0.6
        numel, mom, skip, kw = _case(K, case)
        try:
            lu = LayUp(K, numel, 0.01, mom, 77 + case, 0, skip, tuning=block or None, **kw)
        except LayUpError as e:
            # a thread shape that cannot hold this tile says so at init (tested elsewhere); anything else is a defect
            assert e.code == LAYUP_EINVAL and any(k in block for k in MAY_REFUSE) and "launch_shape" not in block, (block, K, case, e)
            continue
        ref = oracle.Oracle(numel, K, 0.01, mom, 77 + case, 0, skip, **kw)
        gen = torch.Generator(device="cuda").manual_seed(case)
        L = len(numel)
        for l in range(L):
            lu.view(WHAT_X, l).normal_(0, 0.02, generator=gen)
            ref.x[l][:] = lu.view(WHAT_X, l).cpu().numpy()
        for step in range(3):
            grads = []
            for l in range(L):
                lu.view(WHAT_G, l).normal_(0, 1e-2, generator=gen)
                grads.append(lu.view(WHAT_G, l).cpu().numpy())
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
                    assert max_ulp(lu.view(what, l).cpu().numpy(), want) == 0, (block, K, case, step, l, what)
            assert np.array_equal(lu.layup_weights(), ref.w), (block, K, case, step)
        lu.close()
        ran += 1
    assert ran > 0 or any(k in block for k in MAY_REFUSE), (block, K)
    if ran == 0:
        pytest.skip("this thread shape holds none of the tiles of K=%d" % K)
