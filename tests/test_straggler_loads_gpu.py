"""GPU parity of the straggler-mode load paths of the fused update kernel (update_tma.cu):

* the default: exactly the rows a round needs as row-by-row bulk copies, every thread posting the
  bytes of its own copies on the tile's mbarrier;
* layup_tuning.tma2d = 1: the same rows four at a time with cp.async.bulk.tensor.2d.tile::gather4
  (rows the round does not need get an out-of-range index);
* split staging (thread shape 5, the straggler-mode default of launches that are not latency bound
  when the optimiser has state): the last array of (x, g, m, v) through registers.

Every combination must give the bits of the oracle (Alg. 1 with the mask of
PAPER.md:220-229): a skipped replica takes no step and pushes nothing but still receives."""
import numpy as np
import pytest

import oracle
import synth
from _util import max_ulp
from paper_2410_05985_b200 import (FUSED_NEVER, MIX_LOSSY, MIX_PUSHSUM, MIX_SYMMETRIC, OPT_ADAMW, OPT_SGD, WHAT_G,
                                   WHAT_M, WHAT_V, WHAT_X, LayUp)

pytestmark = pytest.mark.gpu

ADAM = dict(weight_decay=0.0031235, beta1=0.9, beta2=0.95, eps=1e-8)
SPLIT = 5            # index of the split-staged thread shape in update_tma.cu's table (include/layup.h: variant)


def _numel(K):
    """Several tiles per layer with ragged tails, a layer smaller than one tile, a one-element layer."""
    per_tile = max(8, 1024 // K) * 4
    return [per_tile * 37 + 5, per_tile * 3 - 1, 1, 33, per_tile * 12]


def _check(K, skip, mu, opt, mix, tuning, rounds=4, delay=(0, 0), per_layer=False):
    numel = _numel(K)
    kw = dict(optimizer=opt, mix_mode=mix, delay_replica=delay[0], delay_rounds=delay[1], **(ADAM if opt == OPT_ADAMW else {}))
    lu = LayUp(K, numel, 3e-3, mu, 91 + K, 0, skip, tuning=tuning, **kw)
    ref = oracle.Oracle(numel, K, 3e-3, mu, 91 + K, 0, skip, **kw)
    w = synth.Workload("t", K, tuple(numel), 3e-3, mu, 0, 91 + K, grad_std=1e-2)
    for l in range(w.L):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
        ref.x[l][:] = lu.view(WHAT_X, l).cpu().numpy()
    idle_seen = False
    for step in range(rounds):
        grads = []
        for l in range(w.L):
            synth.fill_grad_(w, step, l, lu.view(WHAT_G, l))
            grads.append(lu.view(WHAT_G, l).cpu().numpy())
        if per_layer and step % 2:
            for l in reversed(range(w.L)):
                lu.layup_layer_update(step, l)
        else:
            lu.layup_round(step)
        lu.layup_sync()
        ref.round(step, grads)
        _, active = lu.layup_schedule(step)
        idle_seen |= not active.all()
        for l in range(w.L):
            pairs = [(WHAT_X, ref.x[l])] + ([(WHAT_M, ref.m[l])] if ref.m is not None else []) + \
                    ([(WHAT_V, ref.v[l])] if ref.v is not None else [])
            for what, want in pairs:
                assert max_ulp(lu.view(what, l).cpu().numpy(), want) == 0, (step, l, what)
        assert np.array_equal(lu.layup_weights(), ref.w), step
    lu.close()
    return idle_seen


@pytest.mark.parametrize("tma2d", [0, 1, 2])
@pytest.mark.parametrize("K,skip,mu,opt,mix", [
    (2, 0.5, 0.0, OPT_SGD, MIX_PUSHSUM), (5, 0.25, 0.9, OPT_SGD, MIX_PUSHSUM), (8, 0.25, 0.9, OPT_SGD, MIX_LOSSY),
    (16, 0.25, 0.9, OPT_SGD, MIX_PUSHSUM), (16, 0.6, 0.0, OPT_ADAMW, MIX_PUSHSUM), (33, 0.25, 0.0, OPT_SGD, MIX_SYMMETRIC),
    (64, 0.25, 0.0, OPT_SGD, MIX_PUSHSUM), (63, 0.9, 0.9, OPT_SGD, MIX_SYMMETRIC), (100, 0.25, 0.0, OPT_ADAMW, MIX_LOSSY),
    (32, 0.25, 0.9, OPT_SGD, MIX_PUSHSUM), (64, 0.4, 0.9, OPT_SGD, MIX_LOSSY)])
def test_straggler_rows_by_copy_and_by_gather4(K, skip, mu, opt, mix, tma2d):
    """Two-launch path (fused = never, so the grouped kernel reads the device tables) and the default."""
    assert _check(K, skip, mu, opt, mix, dict(tma2d=tma2d, fused=FUSED_NEVER))
    _check(K, skip, mu, opt, mix, dict(tma2d=tma2d), rounds=3, per_layer=True)


@pytest.mark.parametrize("K,skip,mu,opt,mix", [
    (4, 0.0, 0.9, OPT_SGD, MIX_PUSHSUM), (16, 0.25, 0.9, OPT_SGD, MIX_PUSHSUM), (16, 0.0, 0.0, OPT_ADAMW, MIX_SYMMETRIC),
    (8, 0.4, 0.0, OPT_ADAMW, MIX_PUSHSUM), (16, 0.25, 0.0, OPT_SGD, MIX_LOSSY), (7, 0.25, 0.9, OPT_SGD, MIX_SYMMETRIC)])
@pytest.mark.parametrize("tma2d", [0, 1])
def test_split_staging_last_array_through_registers(K, skip, mu, opt, mix, tma2d):
    """Thread shape 5 forced for every launch, with and without idle replicas, every optimiser (SGD
    without momentum stages g through registers, momentum m, AdamW v)."""
    _check(K, skip, mu, opt, mix, dict(variant=SPLIT, tma2d=tma2d))


@pytest.mark.parametrize("K,skip,mu,variant", [(4, 0.0, 0.0, 0), (16, 0.0, 0.0, 0), (16, 0.0, 0.0, 6), (9, 0.3, 0.0, 6),
                                               (32, 0.0, 0.9, 7), (64, 0.25, 0.9, 7), (48, 0.25, 0.9, 7)])
def test_thread_shapes_of_the_launches_that_are_not_latency_bound(K, skip, mu, variant):
    """Shape 6 (six CTAs per SM; the default for SGD without momentum and tiles of <= 1024 items) and
    shape 7 (split staging for tiles of 2048 items; the straggler-mode default for K >= 32 with
    momentum), as the library picks them (variant 0, two-launch path) and forced."""
    _check(K, skip, mu, OPT_SGD, MIX_PUSHSUM, dict(variant=variant, fused=FUSED_NEVER))
    _check(K, skip, mu, OPT_SGD, MIX_SYMMETRIC, dict(variant=variant, fused=FUSED_NEVER), rounds=2)


def test_split_staging_refuses_tiles_it_cannot_hold():
    from paper_2410_05985_b200 import LAYUP_EINVAL, LayUpError
    with pytest.raises(LayUpError) as e:
        LayUp(64, [5000], 0.01, tuning=dict(variant=SPLIT, tile_items=4096))
    assert e.value.code == LAYUP_EINVAL


def test_delay_mode_straggler_takes_the_same_paths():
    """PAPER.md:220 delay-mode straggler (R19): replica 3 is active every third round only."""
    for tma2d in (0, 1):
        assert _check(16, 0.0, 0.9, OPT_SGD, MIX_PUSHSUM, dict(tma2d=tma2d, fused=FUSED_NEVER), rounds=6, delay=(3, 2))
