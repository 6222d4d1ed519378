"""NEXT-1: the paper-faithful trigger.  A real backward pass drives the path:
per-layer gradient hooks call layup_layer_update "as soon as the corresponding gradients for that
layer are available" (Algorithm 1 "Notify updater thread"),
output layer first (Fig. 1), with one peer per iteration (peer_mode 1).

K replicas of a 3-layer MLP (configs[0] shapes) live IN the arena: every replica's weight and bias
are strided torch views of its layer slice, so the forward pass reads the parameters the kernels
write, with no copies.  The paper's datasets are unavailable; the task is a seeded synthetic
teacher-student regression, each worker drawing its own mini-batches.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2410_05985_b200 import WHAT_G, WHAT_X, LayUp

pytestmark = pytest.mark.gpu

DIMS = [(256, 256), (256, 256), (256, 10)]            # (in, out) of configs[0]


def _views(lu, what, K):
    """Per layer: (W[K,out,in], b[K,out]) as strided views of the arena slice [W | b]."""
    out = []
    for l, (din, dout) in enumerate(DIMS):
        v = lu.view(what, l)                           # [K, numel] with row stride = pad
        W = v.as_strided((K, dout, din), (v.stride(0), din, 1), v.storage_offset())
        b = v.as_strided((K, dout), (v.stride(0), 1), v.storage_offset() + din * dout)
        out.append((W, b))
    return out


def _forward(params, X):
    h = X                                              # [K, B, in]
    for l, (W, b) in enumerate(params):
        h = torch.baddbmm(b.unsqueeze(1), h, W.transpose(1, 2))
        if l + 1 < len(params):
            h = torch.relu(h)
    return h


def test_backward_hooks_drive_layerwise_updates():
    K, B, lr, steps, seed = 4, 64, 0.1, 60, 11
    numel = [i * o + o for i, o in DIMS]
    lu = LayUp(K, numel, lr=lr, momentum=0.0, seed=seed, peer_mode=1)
    ref = oracle.Oracle(numel, K, lr=lr, momentum=0.0, seed=seed, peer_mode=1)
    gen = torch.Generator(device="cuda").manual_seed(0)
    for l, (din, dout) in enumerate(DIMS):
        row = torch.randn(numel[l], device="cuda", generator=gen) / np.sqrt(din)
        row[din * dout:] = 0.0                                                 # biases start at zero
        lu.view(WHAT_X, l).copy_(row.unsqueeze(0).expand(K, -1))               # common x0
        ref.x[l][:] = lu.view(WHAT_X, l).cpu().numpy()
    teacher = [((torch.randn(1, o, i, device="cuda", generator=gen) / np.sqrt(i)).expand(K, -1, -1),
                torch.zeros(K, o, device="cuda")) for i, o in DIMS]

    params = _views(lu, WHAT_X, K)
    gviews = _views(lu, WHAT_G, K)
    leaves = []
    for W, b in params:
        # .data: same arena memory, own autograd version counter -- the kernels (and the G-slice copies)
        # write the arena behind autograd's back, exactly like the paper's lock-free updater threads
        leaves.append((W.data.requires_grad_(True), b.data.requires_grad_(True)))

    state = {"step": 0, "pending": [2] * len(DIMS), "order": [], "grads": {}}

    def make_hook(l, which):
        def hook(p):
            # the layer's gradient exists: park it in the arena's G slice ...
            gviews[l][which].copy_(p.grad)
            p.grad = None
            state["pending"][l] -= 1
            if state["pending"][l] == 0:
                # ... and notify the updater: local step + gossip for this layer, now,
                # on the stream the backward pass runs on, while earlier layers are still back-propagating
                state["grads"][l] = lu.view(WHAT_G, l).detach().cpu().numpy().copy()
                lu.layup_layer_update(state["step"], l)
                state["order"].append(l)
        return hook

    for l, (W, b) in enumerate(leaves):
        W.register_post_accumulate_grad_hook(make_hook(l, 0))
        b.register_post_accumulate_grad_hook(make_hook(l, 1))

    def disagreement():
        """sum_i ||x_i - xbar||^2 / (K ||xbar||^2): the model disagreement the paper tracks."""
        d = n = 0.0
        for l in range(len(DIMS)):
            x = lu.view(WHAT_X, l).double()
            d += float(((x - x.mean(0, keepdim=True)) ** 2).sum())
            n += float((x.mean(0) ** 2).sum())
        return d / (K * n)

    losses, dis = [], []
    for step in range(steps):
        state.update(step=step, pending=[2] * len(DIMS), order=[], grads={})
        X = torch.randn(K, B, DIMS[0][0], device="cuda", generator=gen)       # each worker its own batch
        with torch.no_grad():
            Y = _forward(teacher, X)
        loss = ((_forward(leaves, X) - Y) ** 2).mean(dim=(1, 2)).sum()       # each worker its own loss
        loss.backward()
        lu.layup_sync()
        losses.append(float(loss.detach()))
        dis.append(disagreement())
        assert state["order"] == [2, 1, 0], "updates must be issued output layer first (PAPER.md:23)"
        ref.round(step, [state["grads"][l] for l in range(len(DIMS))])
        for l in range(len(DIMS)):
            got = lu.view(WHAT_X, l).cpu().numpy()
            assert np.array_equal(got, ref.x[l]), (step, l)                   # bit-exact against the oracle
    w = lu.layup_weights()
    assert np.array_equal(w, ref.w) and (w == w[0][None, :]).all()            # Alg. 1's scalar w_i (R1)
    assert np.mean(losses[-5:]) < 0.75 * np.mean(losses[:5]), losses          # training makes progress
    assert 0.0 < max(dis) < 1e-2, max(dis)                                    # disagreement stays bounded (eq. 9)
    lu.close()
