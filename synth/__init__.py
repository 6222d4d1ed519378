"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: it only names the workloads of
BASELINE.json:configs (layer shapes, K, lr, momentum, rounds) and fills tensors with
seeded random numbers.  It imports neither oracle/ nor paper_2410_05985_b200/; both
sides receive the bytes produced here.

The paper's own workloads (CIFAR-100 / ImageNet-1k / MiniPile / Wikitext-103 with
trained ResNet / GPT-2 models) are not available; these inputs take
their parameter *shapes* (GPT-2 small / medium tensor lists) and value scales
(init std 0.02, small gradients) and stand in for them.
"""
from dataclasses import dataclass, field, replace
from typing import List, Optional, Tuple

import numpy as np
import torch


def mlp_layers(widths_in_out: List[Tuple[int, int]]) -> List[int]:
    """One layer = weight [in x out] fused with its bias [out] (R13)."""
    return [i * o + o for i, o in widths_in_out]


def gpt2_layers(d: int, ffn: int, vocab: int, ctx: int, blocks: int) -> List[int]:
    """GPT-2 tensor groups in forward order: wte, wpe, per block (ln_1, c_attn, attn.c_proj,
    ln_2, c_fc, mlp.c_proj), ln_f; weights fused with their biases (R13)."""
    out = [vocab * d, ctx * d]
    for _ in range(blocks):
        out += [2 * d, d * 3 * d + 3 * d, d * d + d, 2 * d, d * ffn + ffn, ffn * d + d]
    out.append(2 * d)
    return out


def manysmall_layers(n_layers: int = 40, lo: int = 64, hi: int = 1024, seed: int = 7) -> List[int]:
    """Square widths log-uniform in [lo, hi]: w = floor(lo * (hi/lo)**u), u ~ U[0,1) from
    numpy's default_rng(seed); layer = w*w + w (R16)."""
    u = np.random.default_rng(seed).random(n_layers)
    w = np.floor(lo * (hi / lo) ** u).astype(np.int64)
    return [int(v * v + v) for v in w]


@dataclass(frozen=True)
class Workload:
    name: str
    K: int
    numel: Tuple[int, ...]
    lr: float
    momentum: float
    rounds: int
    seed: int                      # Philox key of the peer selector AND base seed of the data
    init_std: float = 0.02
    grad_std: float = 1e-2
    skip_prob: float = 0.0
    peer_mode: int = 0
    heavy_frac: float = 0.0        # fraction of gradient elements scaled by heavy_scale
    heavy_scale: float = 1.0
    common_init: bool = False      # R12: replicas start independent unless asked otherwise
    note: str = ""

    @property
    def L(self) -> int:
        return len(self.numel)

    @property
    def params_per_replica(self) -> int:
        return int(sum(self.numel))


def workloads() -> List[Workload]:
    """BASELINE.json:configs[0..4], in order."""
    mlp3 = tuple(mlp_layers([(256, 256), (256, 256), (256, 10)]))
    return [
        Workload("mlp3_k4", 4, mlp3, lr=0.01, momentum=0.0, rounds=10, seed=0, grad_std=1e-2,
                 note="configs[0]"),
        Workload("gpt2s_k8", 8, tuple(gpt2_layers(768, 3072, 50257, 1024, 12)), lr=3e-4, momentum=0.9,
                 rounds=20, seed=1, grad_std=1e-3, note="configs[1]"),
        Workload("gpt2m_k16", 16, tuple(gpt2_layers(1024, 4096, 50257, 1024, 24)), lr=1e-4, momentum=0.9,
                 rounds=10, seed=2, grad_std=1e-3, heavy_frac=0.01, heavy_scale=100.0, note="configs[2]"),
        Workload("straggler_k8", 8, mlp3, lr=0.01, momentum=0.0, rounds=50, seed=3, grad_std=1e-2,
                 skip_prob=0.25, note="configs[3]"),
        Workload("manysmall_k64", 64, tuple(manysmall_layers()), lr=0.01, momentum=0.0, rounds=100,
                 seed=4, grad_std=1e-2, note="configs[4]"),
    ]


def workload(which) -> Workload:
    ws = workloads()
    if isinstance(which, int):
        return ws[which]
    for w in ws:
        if w.name == which:
            return w
    raise KeyError(which)


def shrink(w: Workload, numel, **kw) -> Workload:
    """Same hyper-parameters on a smaller layer list (parity-test sizes)."""
    return replace(w, numel=tuple(int(n) for n in numel), **kw)


# ---- seeded fills -------------------------------------------------------------------
_KIND_INIT, _KIND_GRAD, _KIND_TAIL = 1, 2, 3


def _seed(base: int, kind: int, step: int, layer: int) -> int:
    ss = np.random.SeedSequence([int(base) & 0xFFFFFFFF, kind, int(step) & 0xFFFFFFFF, int(layer)])
    return int(ss.generate_state(1, dtype=np.uint64)[0] & np.uint64(0x7FFFFFFFFFFFFFFF))


def _gen(device, seed: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def fill_init_(w: Workload, layer: int, x_layer: torch.Tensor) -> None:
    """x_layer: [K, numel] fp32 view (any device, may be strided). N(0, init_std) i.i.d.;
    independent per replica unless w.common_init (then replica 0's draw is broadcast)."""
    gen = _gen(x_layer.device, _seed(w.seed, _KIND_INIT, 0, layer))
    if w.common_init:
        row = torch.empty(x_layer.shape[1], dtype=torch.float32, device=x_layer.device)
        row.normal_(0.0, w.init_std, generator=gen)
        x_layer.copy_(row.unsqueeze(0).expand_as(x_layer))
    else:
        x_layer.normal_(0.0, w.init_std, generator=gen)


def fill_grad_(w: Workload, step: int, layer: int, g_layer: torch.Tensor, data_seed: Optional[int] = None) -> None:
    """g_layer: [K, numel] fp32 view. N(0, grad_std); if heavy_frac > 0 an independent
    uniform draw scales that fraction of the elements by heavy_scale (R17)."""
    base = w.seed if data_seed is None else data_seed
    g_layer.normal_(0.0, w.grad_std, generator=_gen(g_layer.device, _seed(base, _KIND_GRAD, step, layer)))
    if w.heavy_frac > 0.0:
        gen = _gen(g_layer.device, _seed(base, _KIND_TAIL, step, layer))
        for i in range(g_layer.shape[0]):          # one replica at a time bounds the scratch memory
            row = g_layer[i]
            u = torch.empty(row.shape, dtype=torch.float32, device=row.device)
            u.uniform_(0.0, 1.0, generator=gen)
            row.mul_(torch.where(u < w.heavy_frac, w.heavy_scale, 1.0))


def host_state(w: Workload):
    """(x, grads_fn) on the CPU: x = list of [K, numel] fp32 numpy arrays, grads_fn(step) likewise."""
    xs = []
    for l, n in enumerate(w.numel):
        t = torch.empty((w.K, n), dtype=torch.float32)
        fill_init_(w, l, t)
        xs.append(t.numpy())

    def grads(step: int):
        gs = []
        for l, n in enumerate(w.numel):
            t = torch.empty((w.K, n), dtype=torch.float32)
            fill_grad_(w, step, l, t)
            gs.append(t.numpy())
        return gs

    return xs, grads
