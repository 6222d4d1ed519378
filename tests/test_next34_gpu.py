"""GPU parity for SURVEY.md 8(f) NEXT-3 (AdamW, coupled weight decay) and NEXT-4 (contention-lossy
and symmetric mixers): the CUDA path through the C-ABI against the oracle on the same seeded
bytes, every round, bit-exact schedule and weights, parameters and optimiser state within 1e-6
(and, the two sides sharing the order of fp32 operations, 0 ulp)."""
import os

import numpy as np
import pytest
import torch

import oracle
import synth
from _util import REL_TOL_100, REL_TOL_ROUND, max_ulp, rel_err
from paper_2410_05985_b200 import (ENGINE_LDG, FUSED_AUTO, FUSED_NEVER, SHAPE_GROUPED, SHAPE_PERSISTENT, LAYUP_EINVAL, MIX_LOSSY, MIX_PUSHSUM, MIX_SYMMETRIC, OPT_ADAMW, OPT_SGD, WHAT_G,
                                   WHAT_M, WHAT_V, WHAT_X, LayUp, LayUpError)

pytestmark = pytest.mark.gpu

ADAM = dict(weight_decay=0.0031235, beta1=0.9, beta2=0.95, eps=1e-8)       # PAPER.md:469-480 + GPT-2 betas


def _pair(K, numel, lr, mu, seed, skip, opt, mix, peer_mode=0, shadow=False, tuning=None, **kw):
    lu = LayUp(K, numel, lr, mu, seed, peer_mode, skip, optimizer=opt, mix_mode=mix, tuning=tuning, **kw)
    ref = oracle.Oracle(numel, K, lr, mu, seed, peer_mode, skip, optimizer=opt, mix_mode=mix, **kw)
    sh = oracle.Oracle(numel, K, lr, mu, seed, peer_mode, skip, optimizer=opt, mix_mode=mix, f64=True, **kw) if shadow else None
    w = synth.Workload("t", K, tuple(numel), lr, mu, 0, seed, grad_std=1e-3, heavy_frac=0.01, heavy_scale=100.0)
    for l in range(len(numel)):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
        x0 = lu.view(WHAT_X, l).cpu().numpy()
        ref.x[l][:] = x0
        if sh is not None:
            sh.x[l][:] = x0
    return w, lu, ref, sh


def _run(w, lu, ref, sh, rounds, expect_zero_ulp=True):
    worst_ulp = 0
    for step in range(rounds):
        grads = []
        for l in range(w.L):
            synth.fill_grad_(w, step, l, lu.view(WHAT_G, l))
            grads.append(lu.view(WHAT_G, l).cpu().numpy())
        lu.layup_round(step)
        lu.layup_sync()
        ref.round(step, grads)
        if sh is not None:
            sh.round(step, grads)
        for l in range(w.L):
            pairs = [(WHAT_X, ref.x[l])]
            if ref.m is not None:
                pairs.append((WHAT_M, ref.m[l]))
            if ref.v is not None:
                pairs.append((WHAT_V, ref.v[l]))
            for what, want in pairs:
                got = lu.view(what, l).cpu().numpy()
                assert rel_err(got, want) <= REL_TOL_ROUND, (step, l, what, rel_err(got, want))
                worst_ulp = max(worst_ulp, max_ulp(got, want))
        assert np.array_equal(lu.layup_weights(), ref.w), step
    if sh is not None:
        for l in range(w.L):
            assert rel_err(lu.view(WHAT_X, l).cpu().numpy(), sh.x[l]) <= REL_TOL_100
    if expect_zero_ulp:
        assert worst_ulp == 0, worst_ulp
    return worst_ulp


NUMEL = [515 * 40, 19 * 40, 80, 40 * 120 + 120, 1, 33, 4097]     # several tiles, ragged tails, tiny layers


@pytest.mark.parametrize("K,skip", [(1, 0.0), (2, 0.0), (3, 0.25), (8, 0.0), (16, 0.25), (33, 0.1), (64, 0.0)])
def test_adamw_parity_every_round(K, skip):
    w, lu, ref, sh = _pair(K, NUMEL, 7.5249e-4, 0.0, 11 + K, skip, OPT_ADAMW, MIX_PUSHSUM, shadow=True, **ADAM)
    _run(w, lu, ref, sh, 12)
    lu.close()


@pytest.mark.parametrize("mu,wd", [(0.0, 0.005), (0.9, 0.0001), (0.9, 0.014)])
def test_sgd_weight_decay_parity(mu, wd):
    w, lu, ref, sh = _pair(8, NUMEL, 0.035, mu, 5, 0.25, OPT_SGD, MIX_PUSHSUM, shadow=True, weight_decay=wd)
    _run(w, lu, ref, sh, 12)
    lu.close()


@pytest.mark.parametrize("K,skip,mu", [(2, 0.0, 0.0), (4, 0.0, 0.9), (8, 0.25, 0.9), (16, 0.0, 0.0), (64, 0.1, 0.0)])
@pytest.mark.parametrize("mix", [MIX_LOSSY, MIX_SYMMETRIC])
def test_variant_mixers_parity(K, skip, mu, mix):
    w, lu, ref, sh = _pair(K, NUMEL, 0.01, mu, 3 * K + mix, skip, OPT_SGD, mix, shadow=True)
    _run(w, lu, ref, sh, 15)
    wts = lu.layup_weights()
    if mix == MIX_SYMMETRIC:
        assert np.array_equal(wts, np.full_like(wts, 1.0 / K))               # no push-sum weight moves
    elif K > 2:
        assert (wts.sum(axis=1) < 1.0).any()                                 # contention lost some mass
    lu.close()


@pytest.mark.parametrize("mix", [MIX_LOSSY, MIX_SYMMETRIC])
@pytest.mark.parametrize("peer_mode", [0, 1])
def test_adamw_with_variant_mixers(mix, peer_mode):
    w, lu, ref, sh = _pair(8, NUMEL, 1e-3, 0.0, 21, 0.2, OPT_ADAMW, mix, peer_mode=peer_mode, shadow=True, **ADAM)
    _run(w, lu, ref, sh, 10)
    lu.close()


def test_symmetric_k2_exact_average_and_mean_conservation_on_device():
    K, n = 2, 4099
    lu = LayUp(K, [n], 0.0, 0.0, 9, mix_mode=MIX_SYMMETRIC)
    rng = np.random.default_rng(0)
    x = (rng.integers(-2**16, 2**16, size=(K, n)) / 1024.0).astype(np.float32)
    lu.view(WHAT_X, 0).copy_(torch.from_numpy(x))
    lu.layup_round(0)
    lu.layup_sync()
    got = lu.view(WHAT_X, 0).cpu().numpy()
    want = ((x[0].astype(np.float64) + x[1]) / 2).astype(np.float32)
    assert np.array_equal(got[0], want) and np.array_equal(got[1], want)
    lu.close()
    K = 16
    lu = LayUp(K, [n], 0.0, 0.0, 9, mix_mode=MIX_SYMMETRIC)
    x = rng.normal(0, 1, (K, n)).astype(np.float32)
    lu.view(WHAT_X, 0).copy_(torch.from_numpy(x))
    mean0 = x.astype(np.float64).mean(axis=0)
    prev = lu.layup_disagreement().sum()
    for t in range(30):
        lu.layup_round(t)
        d = lu.layup_disagreement().sum()
        assert d <= prev * (1 + 1e-6)
        prev = d
    got = lu.view(WHAT_X, 0).cpu().numpy().astype(np.float64)
    np.testing.assert_allclose(got.mean(axis=0), mean0, atol=4 * K * 2**-24 * 30)
    lu.close()


def test_layer_calls_equal_round_for_adamw():
    """layup_layer_update on streams, output layer first, == layup_round bit for bit (AdamW state included)."""
    K = 8
    outs = []
    for mode in ("round", "layers"):
        w, lu, ref, _ = _pair(K, NUMEL, 1e-3, 0.0, 4, 0.25, OPT_ADAMW, MIX_PUSHSUM, **ADAM)
        streams = [torch.cuda.Stream() for _ in range(3)]
        for step in range(5):
            for l in range(w.L):
                synth.fill_grad_(w, step, l, lu.view(WHAT_G, l))
            torch.cuda.synchronize()
            if mode == "round":
                lu.layup_round(step)
            else:
                for k, l in enumerate(reversed(range(w.L))):
                    lu.layup_layer_update(step, l, streams[k % 3])
            lu.layup_sync()
        outs.append([lu.view(what, l).cpu().numpy().copy() for l in range(w.L) for what in (WHAT_X, WHAT_M, WHAT_V)])
        lu.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("opt,mix,K", [(OPT_ADAMW, MIX_PUSHSUM, 8), (OPT_ADAMW, MIX_SYMMETRIC, 8), (OPT_SGD, MIX_SYMMETRIC, 16),
                                       (OPT_ADAMW, MIX_PUSHSUM, 500)])
def test_ldg_engine_covers_the_widened_rule(opt, mix, K):
    """The LDG kernels (large K, or layup_tuning.engine = 2) implement the same optimisers and mixers.
    K = 500 with AdamW does not fit the TMA staging and takes the LDG engine by itself."""
    kw = ADAM if opt == OPT_ADAMW else {}
    numel = NUMEL if K < 100 else [4097, 33, 800]
    w, lu, ref, _ = _pair(K, numel, 1e-3, 0.0, 8, 0.2, opt, mix, tuning=dict(engine=ENGINE_LDG) if K < 100 else None, **kw)
    _run(w, lu, ref, None, 6)
    lu.close()


def test_adamw_full_size_sampled_parity():
    """configs[1] shapes (K = 8 GPT-2-small) with AdamW at full size, sampled columns (as
    test_parity_gpu.test_full_size_sampled_parity): 28 B per parameter update."""
    wl = synth.workload("gpt2s_k8")
    free, _ = torch.cuda.mem_get_info()
    need = wl.K * sum((n + 31) // 32 * 32 for n in wl.numel) * 4 * 4
    if need + (8 << 30) > free:
        pytest.skip("needs %.1f GB of HBM" % (need / 2**30))
    lu = LayUp(wl.K, wl.numel, wl.lr, 0.0, wl.seed, optimizer=OPT_ADAMW, **ADAM)
    rng = np.random.default_rng(1)
    from test_parity_gpu import _sample_columns
    cols = [torch.from_numpy(_sample_columns(n, max(8, 1024 // wl.K), rng)).cuda() for n in wl.numel]
    ref = oracle.Oracle([int(c.numel()) for c in cols], wl.K, wl.lr, 0.0, wl.seed, optimizer=OPT_ADAMW, **ADAM)
    for l in range(wl.L):
        synth.fill_init_(wl, l, lu.view(WHAT_X, l))
        ref.x[l][:] = lu.view(WHAT_X, l)[:, cols[l]].cpu().numpy()
    for step in range(3):
        grads = []
        for l in range(wl.L):
            synth.fill_grad_(wl, step, l, lu.view(WHAT_G, l))
            grads.append(lu.view(WHAT_G, l)[:, cols[l]].cpu().numpy())
        lu.layup_round(step)
        lu.layup_sync()
        ref.round(step, grads)
        for l in range(wl.L):
            for what, want in ((WHAT_X, ref.x[l]), (WHAT_M, ref.m[l]), (WHAT_V, ref.v[l])):
                got = lu.view(what, l)[:, cols[l]].cpu().numpy()
                assert rel_err(got, want) <= REL_TOL_ROUND and max_ulp(got, want) == 0, (step, l, what)
        assert np.array_equal(lu.layup_weights(), ref.w)
    lu.close()
    del lu
    torch.cuda.empty_cache()


def test_argument_errors_of_the_new_fields():
    for kw in (dict(optimizer=2), dict(mix_mode=3), dict(weight_decay=-1.0), dict(optimizer=OPT_ADAMW, beta1=1.0),
               dict(optimizer=OPT_ADAMW, eps=-1e-8)):
        with pytest.raises(LayUpError) as e:
            LayUp(4, [100], 0.1, **kw)
        assert e.value.code == LAYUP_EINVAL
    lu = LayUp(4, [100], 0.1)
    with pytest.raises(LayUpError):
        lu.ptr(WHAT_V, 0, 0)                      # no V section without AdamW
    lu.close()
    lu = LayUp(4, [100], 0.1, optimizer=OPT_ADAMW)
    assert lu.view(WHAT_V, 0).shape == (4, 100) and lu.view(WHAT_M, 0).shape == (4, 100)
    lu.close()


@pytest.mark.parametrize("opt,mix,mu,skip", [(OPT_SGD, MIX_PUSHSUM, 0.0, 0.0), (OPT_SGD, MIX_PUSHSUM, 0.9, 0.25),
                                             (OPT_SGD, MIX_LOSSY, 0.9, 0.1), (OPT_SGD, MIX_SYMMETRIC, 0.0, 0.25),
                                             (OPT_ADAMW, MIX_PUSHSUM, 0.0, 0.25), (OPT_ADAMW, MIX_LOSSY, 0.0, 0.0),
                                             (OPT_ADAMW, MIX_SYMMETRIC, 0.0, 0.0)])
@pytest.mark.parametrize("K", [1, 2, 5, 16, 64])
def test_single_launch_path_equals_two_launch_path(opt, mix, mu, skip, K):
    """Launch-latency-bound launches compute the schedule stage inside the update kernel (one
    launch per round / per layer event); larger ones run the schedule kernel first.  Same bits,
    same weights, and both equal the oracle."""
    kw = ADAM if opt == OPT_ADAMW else {}
    outs, launches = [], []
    for fused in (FUSED_AUTO, FUSED_NEVER):
        w, lu, ref, _ = _pair(K, NUMEL, 1e-3, mu, 31, skip, opt, mix, tuning=dict(fused=fused, fused_waves=4), **kw)
        n0 = lu.layup_launch_count()
        _run(w, lu, ref, None, 4)
        # per-layer events take the same path
        for l in range(w.L):
            synth.fill_grad_(w, 4, l, lu.view(WHAT_G, l))
        for l in reversed(range(w.L)):
            lu.layup_layer_update(4, l)
        lu.layup_sync()
        launches.append(lu.layup_launch_count() - n0)
        outs.append([lu.view(WHAT_X, l).cpu().numpy().copy() for l in range(w.L)] + [lu.layup_weights()])
        lu.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)
    assert launches[0] == 4 + len(NUMEL) and launches[1] == 2 * launches[0]


@pytest.mark.parametrize("opt,mix", [(OPT_SGD, MIX_PUSHSUM), (OPT_ADAMW, MIX_PUSHSUM), (OPT_ADAMW, MIX_SYMMETRIC)])
def test_pads_stay_zero_and_nothing_is_written_out_of_bounds(opt, mix):
    """Bounds check of our own (compute-sanitizer is closed on this pool): every slice is padded to
    32 floats; the kernels process the padded length and must leave every pad float of every
    section exactly zero, for ragged sizes on both sides of a tile boundary."""
    K = 8
    numel = [1, 31, 33, 127, 129, 255 * 4 + 1, 4096 + 3, 8191, 1000]
    kw = ADAM if opt == OPT_ADAMW else {}
    lu = LayUp(K, numel, 1e-3, 0.9 if opt == OPT_SGD else 0.0, 2, 0, 0.25, optimizer=opt, mix_mode=mix, **kw)
    n_sec = 4 if opt == OPT_ADAMW else 3
    for step in range(6):
        for l in range(len(numel)):
            lu.view(WHAT_X if step == 0 else WHAT_G, l).normal_(0, 1)
            lu.view(WHAT_G, l).normal_(0, 1)
        if step % 2:
            lu.layup_round(step)
        else:
            for l in reversed(range(len(numel))):
                lu.layup_layer_update(step, l)
        lu.layup_sync()
    for what in range(n_sec):
        for l, n in enumerate(numel):
            pad = (n + 31) // 32 * 32
            p0, _ = lu.ptr(what, 0, l)
            off = (p0 - lu._base) // 4
            full = lu._arena_f32.as_strided((K, pad), (pad, 1), off)
            assert bool((full[:, n:] == 0).all()), (what, l)
            assert bool(torch.isfinite(full).all())
    lu.close()


@pytest.mark.parametrize("opt", [OPT_SGD, OPT_ADAMW])
def test_checkpoint_resume_is_bit_identical(opt):
    """layup_state_export / layup_state_import + a copy of the arena = a resumable snapshot."""
    K = 8
    kw = ADAM if opt == OPT_ADAMW else {}
    mu = 0.9 if opt == OPT_SGD else 0.0
    w, a, _, _ = _pair(K, NUMEL, 1e-3, mu, 17, 0.25, opt, MIX_PUSHSUM, **kw)
    def grads(lu, step):
        for l in range(w.L):
            synth.fill_grad_(w, step, l, lu.view(WHAT_G, l))

    for step in range(4):
        grads(a, step)
        a.layup_round(step)
    # a layer-wise partial round: the three last layers are one step ahead at the snapshot
    grads(a, 4)
    for l in (w.L - 1, w.L - 2, w.L - 3):
        a.layup_layer_update(4, l)
    state = a.layup_state_export()
    b = LayUp(K, NUMEL, 1e-3, mu, 17, 0, 0.25, optimizer=opt, mix_mode=MIX_PUSHSUM, **kw)
    b._arena_f32.copy_(a._arena_f32)
    b.layup_state_import(*state)
    with pytest.raises(LayUpError):
        b.layup_round(4)                              # layers disagree about the step: refused
    for lu in (a, b):
        for l in reversed(range(w.L - 3)):
            lu.layup_layer_update(4, l)
        for step in range(5, 8):
            grads(lu, step)
            lu.layup_round(step)
        lu.layup_sync()
    for what in ([WHAT_X, WHAT_M] + ([WHAT_V] if opt == OPT_ADAMW else [])):
        for l in range(w.L):
            assert torch.equal(a.view(what, l), b.view(what, l)), (what, l)
    assert np.array_equal(a.layup_weights(), b.layup_weights())
    a.close(); b.close()


@pytest.mark.parametrize("K", [1, 3, 8, 16, 64, 100])
@pytest.mark.parametrize("opt,mix,mu,skip", [(OPT_SGD, MIX_PUSHSUM, 0.0, 0.0), (OPT_SGD, MIX_LOSSY, 0.9, 0.0),
                                             (OPT_ADAMW, MIX_PUSHSUM, 0.0, 0.0), (OPT_SGD, MIX_PUSHSUM, 0.9, 0.25),
                                             (OPT_SGD, MIX_SYMMETRIC, 0.0, 0.25), (OPT_ADAMW, MIX_SYMMETRIC, 0.0, 0.0)])
@pytest.mark.parametrize("stages", [0, 2])
def test_persistent_form_equals_grouped_form(K, opt, mix, mu, skip, stages):
    """layup_tuning.launch_shape = 2: resident CTAs drain the work list through a multi-stage TMA ring
    (producer warp + consumer warps).  Same bits as the one-CTA-per-work-item launch and as the oracle,
    for every mixer and for straggler rounds (fused = never keeps these small launches off the
    single-launch path so that the persistent kernel is the one that runs; one CTA per SM forces
    every CTA through many tiles and several layers; stages = 2 is the shallowest ring, the
    default the deepest that fits)."""
    kw = ADAM if opt == OPT_ADAMW else {}
    outs = []
    for shape in (SHAPE_PERSISTENT, SHAPE_GROUPED):
        w, lu, ref, _ = _pair(K, NUMEL + [300000], 1e-3, mu, 61 + K, skip, opt, mix,
                              tuning=dict(launch_shape=shape, fused=FUSED_NEVER, ctas_per_sm=1, stages=stages), **kw)
        _run(w, lu, ref, None, 3)
        outs.append([lu.view(WHAT_X, l).cpu().numpy().copy() for l in range(w.L)] + [lu.layup_weights()])
        lu.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)
