"""layup_disagreement_static: the model-disagreement reduction (PAPER.md:389-395 Fig. A1, eq. (9)
PAPER.md:551) for callers that cannot allocate device memory.

Who cannot: a monitoring hook that fires while the backward pass and earlier layers' gossip are
still running on other streams -- cudaMalloc and cudaFree wait for the whole
device, so one allocation there undoes the overlap LayUp is built on; a job whose HBM is already
handed out in full (arena + a framework's caching allocator); a process that borrows an X section
but never made a ctx (layup_init allocates the library's tables).  For them the library keeps the
kernel's fp64 accumulators and its copy of the weights in a static __device__ array inside
liblayup.so (LAYUP_STATIC_MAX_PAIRS = 16384 (layer, replica) pairs, 256 KiB per GPU), and the
entry point calls no cudaMalloc / cudaFree.

Checked here: the static entry point returns what the ctx-based layup_disagreement returns (same
kernels, scratch in a different place) within the 1e-9 relative bar test_next2_gpu.py uses against
the oracle, on consecutive calls -- the array still holds the previous call's sums and weights, so
a missing clear shows up on the second call -- and it refuses shapes beyond the array.

This file sorts last on purpose (pytest -x stops at the first failure, so a defect here hides
nothing else) and passes alone in a fresh process as well as after the other tests: the per-device
set-up (cudaGetSymbolAddress) happens inside the first call, whenever that is.
"""
import ctypes

import numpy as np
import pytest
import torch

import oracle
import synth
from _util import load_grads
from paper_2410_05985_b200 import (LAYUP_EINVAL, LAYUP_STATIC_MAX_PAIRS, WHAT_X, LayUp, LayUpError,
                                   layup_disagreement_static, load_library)

REL = 1e-9          # of the largest distance of the layer, as in tests/test_next2_gpu.py


def _close(got, want):
    for l in range(want.shape[0]):
        scale = max(want[l].max(), 1e-300)
        assert np.abs(got[l] - want[l]).max() <= REL * scale, (l, got[l], want[l])


@pytest.mark.gpu
@pytest.mark.parametrize("K", [3, 16, 64, 200])       # ring kernel (exact and predicated shapes), general kernel
def test_static_scratch_matches_ctx_path_on_consecutive_calls(K):
    numel = [1, 33, 1000, 4097, 70001 if K <= 16 else 2049]
    w = synth.Workload("noalloc", K, tuple(numel), lr=0.05, momentum=0.0, rounds=2, seed=11 + K, grad_std=1e-2)
    lu = LayUp(w.K, w.numel, w.lr, w.momentum, w.seed)
    for l in range(w.L):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
    x_dev = lu.ptr(WHAT_X, 0, 0)[0]
    calls = 0
    for rounds_done in range(w.rounds + 1):
        lu.layup_sync()
        wts = lu.layup_weights()
        # weighted then plain then weighted again: back-to-back calls that reuse both halves of the array
        for weighted in (True, False, True):
            want = lu.layup_disagreement(weighted)                                        # existing path
            got = layup_disagreement_static(x_dev, K, w.numel, wts if weighted else None)  # first / next call
            again = layup_disagreement_static(x_dev, K, w.numel, wts if weighted else None)  # straight after it
            calls += 2
            _close(got, want)
            _close(again, want)
            for l in range(w.L):                                                          # and both against the oracle
                ref = oracle.disagreement(lu.view(WHAT_X, l).cpu().numpy(), wts[l] if weighted else None)
                assert np.abs(got[l] - ref).max() <= REL * max(ref.max(), 1e-300)
        if rounds_done < w.rounds:
            load_grads(w, lu, rounds_done)
            lu.layup_round(rounds_done)
    # a smaller problem right after a larger one: the tail of the array keeps the old sums, the head is cleared
    small = layup_disagreement_static(lu.ptr(WHAT_X, 0, 0)[0], K, w.numel[:1])
    _close(small, lu.layup_disagreement(False)[:1])
    assert calls == 18
    lu.close()


@pytest.mark.gpu
def test_static_scratch_works_without_any_ctx():
    """A caller that never ran layup_init: its own buffer in the arena layout, plain mean."""
    K, numel = 8, [100, 5000, 31]
    pads = [(n + 31) // 32 * 32 for n in numel]
    buf = torch.zeros(sum(K * p for p in pads) + 32, dtype=torch.float32, device="cuda")
    shift = ((-buf.data_ptr()) % 128) // 4
    g = torch.Generator(device="cuda").manual_seed(1234)
    host, off = [], shift
    for n, p in zip(numel, pads):
        v = buf[off:off + K * p].view(K, p)
        v[:, :n] = torch.randn(K, n, generator=g, device="cuda")
        host.append(v[:, :n].cpu().numpy())
        off += K * p
    torch.cuda.current_stream().synchronize()
    for _ in range(2):
        got = layup_disagreement_static(buf.data_ptr() + 4 * shift, K, numel)
        for l in range(len(numel)):
            ref = oracle.disagreement(host[l], None)
            assert np.abs(got[l] - ref).max() <= REL * ref.max()


def test_static_scratch_refuses_what_it_cannot_hold():
    """Argument errors come back before any CUDA call, so this part needs no GPU."""
    lib = load_library()
    one = (ctypes.c_int64 * 1)(64)
    out = np.zeros(4, dtype=np.float64)
    L = LAYUP_STATIC_MAX_PAIRS // 1024 + 1
    many = (ctypes.c_int64 * L)(*([64] * L))
    big = np.zeros(L * 1024, dtype=np.float64)
    assert lib.layup_disagreement_static(128, 1024, L, many, None, big.ctypes.data, None) == LAYUP_EINVAL
    text = lib.layup_last_error(None).decode()
    assert "LAYUP_STATIC_MAX_PAIRS" in text and str(L * 1024) in text
    assert lib.layup_disagreement_static(None, 4, 1, one, None, out.ctypes.data, None) == LAYUP_EINVAL
    assert lib.layup_disagreement_static(128, 0, 1, one, None, out.ctypes.data, None) == LAYUP_EINVAL
    assert lib.layup_disagreement_static(64, 4, 1, one, None, out.ctypes.data, None) == LAYUP_EINVAL       # misaligned
    with pytest.raises(LayUpError) as e:
        layup_disagreement_static(128, 1024, [64] * L)
    assert e.value.code == LAYUP_EINVAL
