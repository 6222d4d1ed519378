"""GPU parity tests proper: the CUDA path, called through the C-ABI binding, against the
oracle, element by element on the same seeded bytes (pytest -m gpu, on the B200 box).

Bars (BASELINE.json north_star): peer indices, active mask and push-sum weights
bit-exact; fp32 parameters within 1e-6 (scale-relative per layer, R15) after
each round and 1e-5 after 100 rounds.  Both sides take the fp32 arithmetic in the same
order with fused multiply-adds, so the tests also record the max ulp distance.
"""
import numpy as np
import pytest
import torch

import oracle
import synth
from _util import REL_TOL_100, REL_TOL_ROUND, compare, load_grads, make_pair, max_ulp, rel_err
from paper_2410_05985_b200 import (LAYUP_EINVAL, LAYUP_ESTATE, WHAT_G, WHAT_M, WHAT_X, LayUp, LayUpError)

pytestmark = pytest.mark.gpu


def _small_workloads():
    ws = synth.workloads()
    return {
        # configs[0] and configs[3] at their full size
        "mlp3_k4": ws[0],
        "straggler_k8": ws[3],
        # GPT-2-shaped sets shrunk so the oracle finishes in seconds; several tiles + ragged tails
        "gpt2s_k8_small": synth.shrink(ws[1], synth.gpt2_layers(48, 200, 1003, 37, 2)),
        "gpt2m_k16_small": synth.shrink(ws[2], synth.gpt2_layers(40, 168, 515, 19, 2)),
        "manysmall_k64_small": synth.shrink(ws[4], synth.manysmall_layers(12, 8, 96, 7)),
    }


@pytest.mark.parametrize("name", list(_small_workloads()))
def test_round_parity_every_round(name):
    w = _small_workloads()[name]
    lu, ref, shadow = make_pair(w, f64_shadow=True)
    worst = worst_ulp = 0
    for step in range(w.rounds):
        grads = load_grads(w, lu, step)
        peer, active = lu.layup_schedule(step)
        rp, ra = oracle.schedule(w.seed, step, w.L, w.K, w.peer_mode, w.skip_prob)
        assert np.array_equal(peer, rp) and np.array_equal(active, ra)          # bit-exact schedule
        lu.layup_round(step)
        lu.layup_sync()
        ref.round(step, grads)
        shadow.round(step, grads)
        e, u = compare(w, lu, ref, REL_TOL_ROUND, "%s step %d" % (name, step))
        worst, worst_ulp = max(worst, e), max(worst_ulp, u)
        assert np.array_equal(lu.layup_weights(), ref.w)                        # fp64 weights bit-exact
    # against exact arithmetic (fp64 shadow): the 100-round bar of north_star
    for l in range(w.L):
        got = lu.view(WHAT_X, l).cpu().numpy()
        assert rel_err(got, shadow.x[l]) <= REL_TOL_100
    print("%s: worst rel err %.2e, worst ulp %d over %d rounds" % (name, worst, worst_ulp, w.rounds))
    assert worst_ulp == 0, "same op order + FMA on both sides should be bit-identical"
    lu.close()


@pytest.mark.parametrize("name,L,rounds", [("mlp3_k4", 3, 10), ("gpt2s_k8", 75, 20), ("gpt2m_k16", 147, 10),
                                           ("straggler_k8", 3, 50), ("manysmall_k64", 40, 100)])
def test_schedule_bit_exact_full_configs(name, L, rounds):
    """Peer indices and the update schedule of every BASELINE config, every round."""
    w = synth.workload(name)
    assert w.L == L and w.rounds == rounds
    lu = LayUp(w.K, [32] * w.L, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob)   # schedule ignores numel
    for step in range(w.rounds):
        peer, active = lu.layup_schedule(step)
        rp, ra = oracle.schedule(w.seed, step, w.L, w.K, w.peer_mode, w.skip_prob)
        assert np.array_equal(peer, rp) and np.array_equal(active, ra)
    lu.close()


@pytest.mark.parametrize("K", [1, 2, 3, 5, 7, 12, 33, 128, 200])
@pytest.mark.parametrize("mu", [0.0, 0.9])
def test_odd_replica_counts_and_ragged_layers(K, mu):
    numel = [1, 31, 32, 33, 127, 1000, 4097, 70001 if K <= 12 else 2049]
    w = synth.Workload("odd", K, tuple(numel), lr=0.05, momentum=mu, rounds=4, seed=100 + K, grad_std=1e-2,
                       skip_prob=0.2 if K > 2 else 0.0)
    lu, ref, _ = make_pair(w)
    for step in range(w.rounds):
        grads = load_grads(w, lu, step)
        lu.layup_round(step)
        ref.round(step, grads)
        _, u = compare(w, lu, ref, REL_TOL_ROUND, "K=%d step %d" % (K, step))
        assert u == 0
        assert np.array_equal(lu.layup_weights(), ref.w)
    # pads stay zero: the slice stride is a multiple of 32 floats and the tail is never dirtied
    for l, n in enumerate(numel):
        p0, _ = lu.ptr(WHAT_X, 0, l)
        pad = (n + 31) // 32 * 32
        full = lu._arena_f32.as_strided((K, pad), (pad, 1), (p0 - lu._base) // 4)
        assert float(full[:, n:].abs().sum()) == 0.0
    lu.close()


def test_k2_exact_pairwise_average_on_device():
    """north_star: K=2 with zero gradient gives exact pairwise averaging."""
    n = 10_000
    lu = LayUp(2, [n], lr=0.1, momentum=0.0, seed=5)
    x = (torch.randint(-2**16, 2**16, (2, n), device="cuda").float() / 1024.0)
    lu.view(WHAT_X, 0).copy_(x)
    lu.layup_round(0)
    lu.layup_sync()
    want = ((x[0].double() + x[1].double()) / 2).float()
    got = lu.view(WHAT_X, 0)
    assert torch.equal(got[0], want) and torch.equal(got[1], want)
    assert np.array_equal(lu.layup_weights(), [[0.5, 0.5]])
    lu.close()


def test_pure_mix_conserves_weighted_mean_and_contracts():
    """Replica-mean conservation and consensus under repeated mixing, on the device path."""
    K, n = 16, 5000
    lu = LayUp(K, [n], lr=0.01, momentum=0.0, seed=9)
    x = lu.view(WHAT_X, 0)
    x.normal_(0, 1, generator=torch.Generator(device="cuda").manual_seed(1))
    w0 = torch.full((K,), 1.0 / K, dtype=torch.float64, device="cuda")
    mean0 = (w0[:, None] * x.double()).sum(0)
    d_prev = None
    for step in range(60):
        lu.layup_round(step)
        wt = torch.from_numpy(lu.layup_weights()[0]).cuda()
        assert abs(float(wt.sum()) - 1.0) < 1e-14
        mean = (wt[:, None] * x.double()).sum(0)
        assert float((mean - mean0).abs().max()) < 4 * K * 2.0 ** -24 * 5 * (1 + step / 20)
        d = float((wt[:, None] * (x.double() - mean[None, :]) ** 2).sum())
        if d_prev is not None:
            # monotone until the fp32 rounding floor (~ n * (2^-24 |x|)^2) is reached
            assert d <= d_prev * (1 + 1e-6) + 1e-10 * n
        d_prev = d
    assert d_prev < 1e-6 * n
    lu.close()


@pytest.mark.parametrize("mode", [0, 1])
def test_layer_calls_on_streams_equal_one_round(mode):
    """I9: layup_round == L calls of layup_layer_update in any order on any streams, bit for bit;
    peer_mode 1 keeps every row of w identical (Algorithm 1's scalar w_i)."""
    base = synth.shrink(synth.workload("gpt2s_k8"), synth.gpt2_layers(32, 128, 301, 16, 2), peer_mode=mode,
                        skip_prob=0.25)
    lu_a, ref, _ = make_pair(base)
    lu_b, _, _ = make_pair(base)
    streams = [torch.cuda.Stream() for _ in range(3)]
    rng = np.random.default_rng(0)
    for step in range(6):
        grads = load_grads(base, lu_a, step)
        for l in range(base.L):
            lu_b.view(WHAT_G, l).copy_(lu_a.view(WHAT_G, l))
        torch.cuda.synchronize()
        lu_a.layup_round(step)
        order = list(reversed(range(base.L))) if step % 2 == 0 else list(rng.permutation(base.L))
        for k, l in enumerate(order):
            lu_b.layup_layer_update(step, int(l), streams[k % 3])
        lu_a.layup_sync()
        lu_b.layup_sync()
        ref.round(step, grads)
        for l in range(base.L):
            assert torch.equal(lu_a.view(WHAT_X, l), lu_b.view(WHAT_X, l))
            assert torch.equal(lu_a.view(WHAT_M, l), lu_b.view(WHAT_M, l))
        assert np.array_equal(lu_a.layup_weights(), lu_b.layup_weights())
        compare(base, lu_a, ref)
        if mode == 1:
            wts = lu_a.layup_weights()
            assert (wts == wts[0][None, :]).all()
    lu_a.close()
    lu_b.close()


@pytest.mark.parametrize("skip", [0.0, 0.25])
def test_persistent_layer_calls_on_streams(skip):
    """The persistent ring (launch_shape = 2) under per-layer events on several streams: every launch
    draws its tiles from the ticket of its own work-list position, so events of different layers that
    overlap on the GPU cannot take or re-arm each other's counter (a shared ticket made tiles run twice
    or not at all).  Layers large enough that the three streams' kernels are resident together;
    fused = never keeps every event on the ring kernel.  Bit for bit against the oracle and against
    one layup_round of the grouped shape."""
    from paper_2410_05985_b200 import FUSED_NEVER, SHAPE_PERSISTENT, LayUp
    numel = [1500000, 999999, 2000003, 1200000, 640000, 1800000, 77]
    w = synth.Workload("ps_streams", 8, tuple(numel), lr=0.01, momentum=0.9, rounds=5, seed=404, skip_prob=skip)
    lu_a, ref, _ = make_pair(w)
    lu_b = LayUp(w.K, w.numel, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob,
                 tuning=dict(launch_shape=SHAPE_PERSISTENT, fused=FUSED_NEVER))
    for l in range(w.L):
        lu_b.view(WHAT_X, l).copy_(lu_a.view(WHAT_X, l))
    streams = [torch.cuda.Stream() for _ in range(3)]
    rng = np.random.default_rng(1)
    for step in range(w.rounds):
        grads = load_grads(w, lu_a, step)
        for l in range(w.L):
            lu_b.view(WHAT_G, l).copy_(lu_a.view(WHAT_G, l))
        torch.cuda.synchronize()
        lu_a.layup_round(step)
        order = list(reversed(range(w.L))) if step % 2 == 0 else list(rng.permutation(w.L))
        for k, l in enumerate(order):
            lu_b.layup_layer_update(step, int(l), streams[k % 3])
        lu_a.layup_sync()
        lu_b.layup_sync()
        ref.round(step, grads)
        for l in range(w.L):
            assert torch.equal(lu_a.view(WHAT_X, l), lu_b.view(WHAT_X, l)), (step, l)
            assert torch.equal(lu_a.view(WHAT_M, l), lu_b.view(WHAT_M, l)), (step, l)
        assert np.array_equal(lu_a.layup_weights(), lu_b.layup_weights())
        _, u = compare(w, lu_b, ref)
        assert u == 0
    lu_a.close()
    lu_b.close()


def test_straggler_semantics_on_device():
    """An inactive replica's x changes iff it received a push; its momentum never changes."""
    w = synth.shrink(synth.workload("straggler_k8"), [5000, 77], momentum=0.9)
    lu, ref, _ = make_pair(w)
    for step in range(20):
        load_grads(w, lu, step)
        peer, active = lu.layup_schedule(step)
        xb = [lu.view(WHAT_X, l).clone() for l in range(w.L)]
        mb = [lu.view(WHAT_M, l).clone() for l in range(w.L)]
        lu.layup_round(step)
        lu.layup_sync()
        for l in range(w.L):
            for i in range(w.K):
                if active[i]:
                    continue
                assert torch.equal(lu.view(WHAT_M, l)[i], mb[l][i])
                received = any(active[s] and peer[l][s] == i for s in range(w.K))
                assert torch.equal(lu.view(WHAT_X, l)[i], xb[l][i]) != received
    lu.close()


def test_host_buffer_round_matches_device_round():
    """layup_round_host (pinned host grads in, params out, layer-pipelined) == layup_round."""
    w = synth.shrink(synth.workload("gpt2s_k8"), synth.gpt2_layers(32, 128, 301, 16, 2))
    lu_a, ref, _ = make_pair(w)
    lu_b, _, _ = make_pair(w)
    total = w.K * sum(w.numel)
    g_host = torch.empty(total, dtype=torch.float32).pin_memory()
    x_host = torch.empty(total, dtype=torch.float32).pin_memory()
    for step in range(3):
        grads = load_grads(w, lu_a, step)
        g_host.copy_(torch.from_numpy(np.concatenate([g.reshape(-1) for g in grads])))
        lu_a.layup_round(step)
        lu_a.layup_sync()
        lu_b.layup_round_host(step, g_host, x_host)
        ref.round(step, grads)
        off = 0
        for l, n in enumerate(w.numel):
            got = x_host[off:off + w.K * n].view(w.K, n)
            assert torch.equal(got, lu_a.view(WHAT_X, l).cpu())
            assert rel_err(got.numpy(), ref.x[l]) <= REL_TOL_ROUND
            off += w.K * n
    lu_a.close()
    lu_b.close()


def test_state_and_argument_errors():
    lu = LayUp(4, [100, 200], lr=0.01)
    with pytest.raises(LayUpError) as e:
        lu.layup_round(1)                       # first round must be step 0
    assert e.value.code == LAYUP_ESTATE
    lu.layup_layer_update(0, 1)
    with pytest.raises(LayUpError) as e:
        lu.layup_layer_update(0, 1)             # (step, layer) applied twice
    assert e.value.code == LAYUP_ESTATE
    with pytest.raises(LayUpError) as e:
        lu.layup_round(0)                       # layer 1 is already past step 0
    assert e.value.code == LAYUP_ESTATE
    lu.layup_layer_update(0, 0)
    lu.layup_round(1)
    with pytest.raises(LayUpError) as e:
        lu.layup_layer_update(2, 5)
    assert e.value.code == LAYUP_EINVAL
    with pytest.raises(LayUpError) as e:
        lu.ptr(WHAT_M, 0, 0)                    # no momentum section in this arena
    assert e.value.code == LAYUP_EINVAL
    lu.layup_sync()
    lu.close()


def _sample_columns(n, C4, rng, n_random=6, width=64):
    """Element indices to check in a big layer: head, ragged tail, and windows straddling
    tile boundaries (tile = C4 float4 columns = 4*C4 floats per replica)."""
    tile = 4 * C4
    idx = [np.arange(0, min(width, n)), np.arange(max(0, n - width), n)]
    n_tiles = (n + tile - 1) // tile
    for t in rng.integers(1, max(2, n_tiles), size=n_random):
        lo = max(0, min(n - 1, int(t) * tile - width // 2))
        idx.append(np.arange(lo, min(n, lo + width)))
    return np.unique(np.concatenate(idx))


# gpt2s_k8 and manysmall_k64 at full size are covered element by element, every configured round, in
# tests/test_fullsize_gpu.py::test_every_element_every_configured_round_full_size
@pytest.mark.parametrize("name,rounds", [("gpt2m_k16", 2)])
def test_full_size_sampled_parity(name, rounds):
    """BASELINE's full sizes in the launch configuration bench.py times (layup_round): the
    update is elementwise in the element index, so the oracle can compute any sampled set of
    columns exactly -- same schedule (keyed on the true layer index), same bytes."""
    w = synth.workload(name)
    free, _ = torch.cuda.mem_get_info()
    need = w.K * sum((n + 31) // 32 * 32 for n in w.numel) * 4 * 3
    if need + (8 << 30) > free:
        pytest.skip("needs %.1f GB of HBM" % (need / 2**30))
    lu = LayUp(w.K, w.numel, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob)
    rng = np.random.default_rng(1)
    C4 = max(8, 1024 // w.K)
    cols = [torch.from_numpy(_sample_columns(n, C4, rng)).cuda() for n in w.numel]
    ref = oracle.Oracle([int(c.numel()) for c in cols], w.K, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob)
    for l in range(w.L):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
        ref.x[l][:] = lu.view(WHAT_X, l)[:, cols[l]].cpu().numpy()
    for step in range(rounds):
        grads = []
        for l in range(w.L):
            synth.fill_grad_(w, step, l, lu.view(WHAT_G, l))
            grads.append(lu.view(WHAT_G, l)[:, cols[l]].cpu().numpy())
        # untouched-by-construction check material: checksum of a replica that is idle this round
        lu.layup_round(step)
        lu.layup_sync()
        ref.round(step, grads)
        for l in range(w.L):
            got = lu.view(WHAT_X, l)[:, cols[l]].cpu().numpy()
            assert rel_err(got, ref.x[l]) <= REL_TOL_ROUND, (name, step, l)
            assert max_ulp(got, ref.x[l]) == 0
            if w.momentum != 0.0:
                gm = lu.view(WHAT_M, l)[:, cols[l]].cpu().numpy()
                assert max_ulp(gm, ref.m[l]) == 0
        assert np.array_equal(lu.layup_weights(), ref.w)
    # a property that holds at any size: every value is finite and the pads are still zero
    for l in (0, w.L - 1):
        assert bool(torch.isfinite(lu.view(WHAT_X, l)).all())
    lu.close()
    del lu
    torch.cuda.empty_cache()


def test_maximum_replica_count():
    """K = LAYUP_MAX_K = 1024 replicas (the LDG kernels take over when the tile of all K replicas no
    longer fits the TMA staging): schedule, weights and parameters against the oracle."""
    K, numel = 1024, [700, 33, 2049]
    w = synth.Workload("kmax", K, tuple(numel), 0.01, 0.9, 3, 77, grad_std=1e-2, skip_prob=0.1)
    lu, ref, _ = make_pair(w)
    for step in range(3):
        grads = load_grads(w, lu, step)
        peer, active = lu.layup_schedule(step)
        rp, ra = oracle.schedule(w.seed, step, w.L, w.K, w.peer_mode, w.skip_prob)
        assert np.array_equal(peer, rp) and np.array_equal(active, ra)
        lu.layup_round(step)
        lu.layup_sync()
        ref.round(step, grads)
        _, u = compare(w, lu, ref, REL_TOL_ROUND, "K=1024 step %d" % step)
        assert u == 0
        assert np.array_equal(lu.layup_weights(), ref.w)
    lu.close()
    with pytest.raises(LayUpError) as e:
        LayUp(1025, [10], 0.1)
    assert e.value.code == LAYUP_EINVAL


def test_layer_larger_than_2_to_31_elements():
    """64-bit indexing: one layer of 2^31 + 1000 elements per replica (8.6 GB), K = 2, sampled
    columns around the start, the 2^31 boundary and the ragged tail against the oracle."""
    n = (1 << 31) + 1000
    free, _ = torch.cuda.mem_get_info()
    if 2 * 2 * (n + 32) * 4 + (6 << 30) > free:
        pytest.skip("needs 35 GB of HBM")
    K = 2
    lu = LayUp(K, [n, 100], 0.5, 0.0, 5)
    cols = torch.cat([torch.arange(0, 300), torch.arange((1 << 31) - 300, (1 << 31) + 300), torch.arange(n - 300, n),
                      torch.arange(3 * (1 << 29) - 50, 3 * (1 << 29) + 50)]).cuda()
    ref = oracle.Oracle([int(cols.numel()), 100], K, 0.5, 0.0, 5)
    x = lu.view(WHAT_X, 0)
    for i in range(K):                                   # cheap deterministic fill of 8.6 GB per replica
        x[i].copy_(torch.arange(n, device="cuda", dtype=torch.float32).mul_(1e-9 * (i + 1)))
    lu.view(WHAT_X, 1).normal_(0, 1)
    ref.x[0][:] = x[:, cols].cpu().numpy()
    ref.x[1][:] = lu.view(WHAT_X, 1).cpu().numpy()
    for step in range(2):
        g = lu.view(WHAT_G, 0)
        for i in range(K):
            g[i].copy_(torch.arange(n, device="cuda", dtype=torch.float32).mul_(1e-10 * (step + 1) * (i + 2)))
        lu.view(WHAT_G, 1).normal_(0, 1)
        grads = [g[:, cols].cpu().numpy(), lu.view(WHAT_G, 1).cpu().numpy()]
        lu.layup_round(step)
        lu.layup_sync()
        ref.round(step, grads)
        assert max_ulp(x[:, cols].cpu().numpy(), ref.x[0]) == 0
        assert max_ulp(lu.view(WHAT_X, 1).cpu().numpy(), ref.x[1]) == 0
    lu.close()
    del lu, x, g
    torch.cuda.empty_cache()


def test_device_schedule_against_curand_directly(curand_pin):
    """The kernels' own Philox pinned to cuRAND's library routine without going through the oracle:
    peers and straggler mask drawn ON THE DEVICE (layup_schedule) must equal the values derived from
    curand_Philox4x32_10 for counter (step, layer | 0xFFFFFFFF, replica, tag) and key = seed."""
    def words(seed, ctrs):
        ctr = np.ascontiguousarray(ctrs, dtype=np.uint32)
        key = np.tile(np.array([seed & 0xFFFFFFFF, seed >> 32], dtype=np.uint32), (ctr.shape[0], 1))
        out = np.empty_like(ctr)
        curand_pin.curand_philox_host(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, ctr.shape[0])
        return out[:, 0].astype(np.uint64)

    for K, L, seed, p, mode in [(8, 5, 0x1234567_89ABCDEF, 0.25, 0), (64, 3, 7, 0.0, 0), (33, 4, 2**63 + 11, 0.5, 1)]:
        lu = LayUp(K, [64] * L, 0.1, 0.0, seed, mode, p)
        thr = min(int(float(np.float32(p)) * 4294967296.0), 0xFFFFFFFF)
        for step in (0, 1, 77, 2**32 - 1):
            peer, active = lu.layup_schedule(step)
            skip = words(seed, [(step, 0xFFFFFFFF, i, 1) for i in range(K)])
            want_active = (skip >= thr) if p > 0 else np.ones(K, dtype=bool)
            assert np.array_equal(active.astype(bool), want_active)
            for l in range(L):
                r = words(seed, [(step, l if mode == 0 else 0xFFFFFFFF, i, 0) for i in range(K)])
                q = (r * np.uint64(K - 1)) >> np.uint64(32)
                want = (q + (q >= np.arange(K, dtype=np.uint64))).astype(np.int64)
                want = np.where(want_active, want, -1)
                assert np.array_equal(peer[l].astype(np.int64), want), (K, step, l)
        lu.close()
