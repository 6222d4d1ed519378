"""Shared helpers of the parity tests: drive the CUDA path (through the C-ABI binding) and
the oracle on the same seeded bytes and compare.  Inputs always flow synth -> both sides;
nothing the CUDA path computes is ever fed to the oracle."""
import numpy as np
import torch

import oracle
import synth
from paper_2410_05985_b200 import WHAT_G, WHAT_M, WHAT_X, LayUp

REL_TOL_ROUND = 1e-6     # BASELINE.json north_star: max relative error after each round
REL_TOL_100 = 1e-5       # ... and after 100 rounds


def rel_err(got, ref):
    """DESIGN.md R15: per layer, max_e |got - ref| / max_e |ref|."""
    scale = float(np.abs(ref).max())
    return float(np.abs(got.astype(np.float64) - ref.astype(np.float64)).max()) / (scale if scale > 0 else 1.0)


def max_ulp(a, b):
    ai = a.view(np.int32).astype(np.int64)
    bi = b.view(np.int32).astype(np.int64)
    ai = np.where(ai < 0, -(ai & 0x7FFFFFFF), ai)
    bi = np.where(bi < 0, -(bi & 0x7FFFFFFF), bi)
    return int(np.abs(ai - bi).max()) if a.size else 0


def make_pair(w, f64_shadow=False, device=0):
    lu = LayUp(w.K, w.numel, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob, device=device)
    ref = oracle.Oracle(w.numel, w.K, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob)
    shadow = oracle.Oracle(w.numel, w.K, w.lr, w.momentum, w.seed, w.peer_mode, w.skip_prob, f64=True) if f64_shadow else None
    for l in range(w.L):
        synth.fill_init_(w, l, lu.view(WHAT_X, l))
        x0 = lu.view(WHAT_X, l).cpu().numpy()
        ref.x[l][:] = x0
        if shadow is not None:
            shadow.x[l][:] = x0
    return lu, ref, shadow


def load_grads(w, lu, step):
    """Fill the arena's G section for `step` and return the same bytes on the host."""
    out = []
    for l in range(w.L):
        synth.fill_grad_(w, step, l, lu.view(WHAT_G, l))
        out.append(lu.view(WHAT_G, l).cpu().numpy())
    return out


def compare(w, lu, ref, tol=REL_TOL_ROUND, tag=""):
    worst, worst_ulp = 0.0, 0
    for l in range(w.L):
        got = lu.view(WHAT_X, l).cpu().numpy()
        e = rel_err(got, ref.x[l])
        assert e <= tol, "%s layer %d rel err %.3e > %.1e" % (tag, l, e, tol)
        worst = max(worst, e)
        worst_ulp = max(worst_ulp, max_ulp(got, ref.x[l]))
        if w.momentum != 0.0:
            gm = lu.view(WHAT_M, l).cpu().numpy()
            assert rel_err(gm, ref.m[l]) <= tol, "%s layer %d momentum" % (tag, l)
            worst_ulp = max(worst_ulp, max_ulp(gm, ref.m[l]))
    return worst, worst_ulp
