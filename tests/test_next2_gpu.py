"""GPU parity for SURVEY 8(f) NEXT-2: delay-mode straggler (DESIGN R19) and the
on-device model-disagreement diagnostic (eq. (9)) against the oracle."""
import time

import numpy as np
import pytest
import torch

import oracle
import synth
from _util import compare, load_grads, max_ulp
from paper_2410_05985_b200 import WHAT_G, WHAT_M, WHAT_X, LayUp

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("K,r,n,p", [(8, 3, 4, 0.0), (4, 0, 1, 0.0), (16, 15, 7, 0.25)])
def test_delay_mode_parity(K, r, n, p):
    w = synth.Workload("delay", K, (5000, 333, 64), lr=0.01, momentum=0.9, rounds=24, seed=77, skip_prob=p)
    lu = LayUp(w.K, w.numel, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob, delay_replica=r, delay_rounds=n)
    ref = oracle.Oracle(w.numel, w.K, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob,
                        delay_replica=r, delay_rounds=n)
    for l in range(w.L):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
        ref.x[l][:] = lu.view(WHAT_X, l).cpu().numpy()
    for step in range(w.rounds):
        grads = load_grads(w, lu, step)
        peer, active = lu.layup_schedule(step)
        rp, ra = oracle.schedule(w.seed, step, w.L, w.K, w.peer_mode, w.skip_prob, r, n)
        assert np.array_equal(peer, rp) and np.array_equal(active, ra)
        if p == 0.0:
            assert active[r] == (1 if (step + 1) % (n + 1) == 0 else 0) and active.sum() >= K - 1
        mb = lu.view(WHAT_M, 0)[r].clone()
        lu.layup_round(step)
        ref.round(step, grads)
        _, u = compare(w, lu, ref)
        assert u == 0
        assert np.array_equal(lu.layup_weights(), ref.w)
        if not active[r]:
            assert torch.equal(lu.view(WHAT_M, 0)[r], mb)         # the straggler took no step of its own
    lu.close()


# 33 ... 63: the split form of the ring kernel (eight lane groups per column block), exact and predicated K
@pytest.mark.parametrize("K", [1, 2, 3, 8, 16, 33, 40, 47, 48, 56, 63, 64, 200, 1000])
def test_disagreement_parity(K):
    numel = [1, 33, 1000, 4097, 70001 if K <= 16 else 2049]
    w = synth.Workload("dis", K, tuple(numel), lr=0.05, momentum=0.0, rounds=3, seed=5 + K, grad_std=1e-2)
    lu = LayUp(w.K, w.numel, w.lr, w.momentum, w.seed)
    for l in range(w.L):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
    for rounds_done in range(w.rounds + 1):
        wts = lu.layup_weights()
        for weighted in (False, True):
            got = lu.layup_disagreement(weighted)
            for l in range(w.L):
                x = lu.view(WHAT_X, l).cpu().numpy()
                want = oracle.disagreement(x, wts[l] if weighted else None)
                scale = max(want.max(), 1e-300)
                assert np.abs(got[l] - want).max() <= 1e-9 * scale, (K, l, weighted, got[l], want)
        if rounds_done < w.rounds:
            load_grads(w, lu, rounds_done)
            lu.layup_round(rounds_done)
    # consensus: identical replicas -> (numerically) zero disagreement
    for l in range(w.L):
        lu.view(WHAT_X, l).copy_(lu.view(WHAT_X, l)[0:1].expand(K, -1).clone())
    d = lu.layup_disagreement(False)
    assert d.max() <= 1e-25
    lu.close()


def test_disagreement_full_size_and_bandwidth():
    """configs[2] shapes: oracle on sampled layers, torch fp64 on the largest layer, and the
    kernel's read bandwidth (4 B per parameter)."""
    w = synth.workload("gpt2m_k16")
    free, _ = torch.cuda.mem_get_info()
    if w.K * w.params_per_replica * 4 * 3 + (24 << 30) > free:
        pytest.skip("needs the configs[2] arena")
    lu = LayUp(w.K, w.numel, w.lr, w.momentum, w.seed)
    for l in range(w.L):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
        synth.fill_grad_(w, 0, l, lu.view(WHAT_G, l))
    for step in range(2):
        lu.layup_round(step)
    lu.layup_sync()
    wts = lu.layup_weights()
    for weighted in (False, True):
        got = lu.layup_disagreement(weighted)
        for l in (w.L - 1, 1, w.L - 6, 3):                    # ln_f, wpe, a c_attn, block-0 c_attn
            want = oracle.disagreement(lu.view(WHAT_X, l).cpu().numpy(), wts[l] if weighted else None)
            assert np.abs(got[l] - want).max() <= 1e-9 * want.max(), (l, weighted)
        x = lu.view(WHAT_X, 0).double()                       # wte, 51.5 M x 16
        c = torch.from_numpy(wts[0]).cuda() if weighted else torch.full((w.K,), 1.0 / w.K, dtype=torch.float64, device="cuda")
        want0 = ((x - (c[:, None] * x).sum(0, keepdim=True)) ** 2).sum(1).cpu().numpy()
        del x
        assert np.abs(got[0] - want0).max() <= 1e-9 * want0.max()
    ms = []
    for _ in range(5):
        lu.layup_disagreement(False)
        ms.append(lu.layup_disagreement_ms())           # device time of the reduction kernels (CUDA events)
    dt = float(np.median(ms)) * 1e-3
    gbs = 4.0 * w.K * w.params_per_replica / dt / 1e9
    print("layup_disagreement on configs[2]: %.3f ms per call on the device, %.0f GB/s read" % (dt * 1e3, gbs))
    assert gbs > 4500
    lu.close()


def test_disagreement_bandwidth_k64():
    """configs[4] shapes (K = 64, 40 layers of 4 K ... 1 M elements): the split form's read rate, and its
    distances against the oracle on every layer."""
    w = synth.workload("manysmall_k64")
    lu = LayUp(w.K, w.numel, w.lr, w.momentum, w.seed)
    for l in range(w.L):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
        synth.fill_grad_(w, 0, l, lu.view(WHAT_G, l))
    lu.layup_round(0)
    lu.layup_sync()
    wts = lu.layup_weights()
    for weighted in (False, True):
        got = lu.layup_disagreement(weighted)
        for l in range(w.L):
            want = oracle.disagreement(lu.view(WHAT_X, l).cpu().numpy(), wts[l] if weighted else None)
            assert np.abs(got[l] - want).max() <= 1e-9 * want.max(), (l, weighted)
    ms = []
    for _ in range(9):
        lu.layup_disagreement(False)
        ms.append(lu.layup_disagreement_ms())
    dt = float(np.median(ms)) * 1e-3
    gbs = 4.0 * w.K * w.params_per_replica / dt / 1e9
    print("layup_disagreement on configs[4]: %.3f ms per call on the device, %.0f GB/s read" % (dt * 1e3, gbs))
    assert gbs > 4800            # measured 5370 (round 2's one-column-per-thread form: 4300)
    lu.close()
