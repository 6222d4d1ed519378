"""ctypes wrapper around oracle/layup_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_2410_05985_b200 and the
product imports nothing from here.  Every function is argument marshalling around
the C file; the arithmetic of the method (Algorithm 1) lives only
in layup_oracle.c.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "layup_oracle.c")
_SO = os.path.join(_HERE, "liblayup_oracle.so")
_lib = None


_CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]


def _compile(so, extra):
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
        tmp = so + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc"] + _CFLAGS + extra + ["-o", tmp, _SRC, "-lm"])
        os.replace(tmp, so)
    return so


def build(force=False):
    """gcc -O2 -ffp-contract=off: no contraction the source does not spell as fmaf()."""
    if force and os.path.exists(_SO):
        os.remove(_SO)
    return _compile(_SO, [])


def build_omp():
    """The same source and flags plus -fopenmp: the element loops marked ORACLE_PAR run on all host
    cores (bench.py's all-cores baseline).  Bit-identical to the serial build (tests/test_oracle_omp.py)."""
    return _compile(os.path.join(_HERE, "liblayup_oracle_omp.so"), ["-fopenmp"])


def _declare(L):
    c = ctypes
    _lib = L
    _lib.oracle_philox4x32_10.argtypes = [c.c_void_p, c.c_void_p, c.c_void_p]
    _lib.oracle_philox4x32_10.restype = None
    _lib.oracle_active.argtypes = [c.c_uint64, c.c_int64, c.c_int32, c.c_float]
    _lib.oracle_active.restype = c.c_int32
    _lib.oracle_peer.argtypes = [c.c_uint64, c.c_int64, c.c_int32, c.c_int32, c.c_int32, c.c_int32]
    _lib.oracle_peer.restype = c.c_int32
    _lib.oracle_active_ex.argtypes = [c.c_uint64, c.c_int64, c.c_int32, c.c_float, c.c_int32, c.c_int32]
    _lib.oracle_active_ex.restype = c.c_int32
    _lib.oracle_schedule.argtypes = [c.c_uint64, c.c_int64, c.c_int32, c.c_int32, c.c_int32, c.c_float,
                                     c.c_int32, c.c_int32, c.c_void_p, c.c_void_p]
    _lib.oracle_disagreement.argtypes = [c.c_int32, c.c_int64, c.c_void_p, c.c_void_p, c.c_void_p]
    _lib.oracle_disagreement.restype = None
    _lib.oracle_schedule.restype = None
    for name, ft in (("oracle_layer_update", c.c_float), ("oracle_layer_update_f64", c.c_double)):
        f = getattr(_lib, name)
        f.argtypes = [c.c_int32, c.c_int64, c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p,
                      ft, ft, c.c_uint64, c.c_int64, c.c_int32, c.c_int32, c.c_float, c.c_int32, c.c_int32,
                      c.c_void_p, c.c_void_p]
        f.restype = c.c_int
    for name in ("oracle_layer_update_ex", "oracle_layer_update_ex_f64"):
        f = getattr(_lib, name)
        f.argtypes = [c.c_int32, c.c_int64, c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p,
                      c.c_void_p, c.c_void_p, c.POINTER(_Opts), c.c_uint64, c.c_int64, c.c_int32, c.c_int32,
                      c.c_float, c.c_int32, c.c_int32, c.c_void_p, c.c_void_p]
        f.restype = c.c_int
    _lib.oracle_mix_tables.argtypes = [c.c_int32, c.c_void_p, c.c_void_p, c.c_void_p, c.c_int32,
                                       c.c_void_p, c.c_void_p, c.c_void_p, c.c_void_p]
    _lib.oracle_mix_tables.restype = None
    return L


def lib():
    global _lib
    if _lib is None:
        _lib = _declare(ctypes.CDLL(build()))
    return _lib


_lib_omp = None


def use_omp(enable=True):
    """Route this module's calls through the -fopenmp build of the same source (or back)."""
    global _lib, _lib_omp
    if enable:
        if _lib_omp is None:
            _lib_omp = _declare(ctypes.CDLL(build_omp()))
        _lib = _lib_omp
    else:
        _lib = None
        lib()


class _Opts(ctypes.Structure):
    """oracle_opts of layup_oracle.c (doubles holding fp32-representable values)."""
    _fields_ = [("optimizer", ctypes.c_int32), ("mix_mode", ctypes.c_int32), ("lr", ctypes.c_double),
                ("mu", ctypes.c_double), ("wd", ctypes.c_double), ("beta1", ctypes.c_double),
                ("beta2", ctypes.c_double), ("eps", ctypes.c_double)]


OPT_SGD, OPT_ADAMW = 0, 1
MIX_PUSHSUM, MIX_LOSSY, MIX_SYMMETRIC = 0, 1, 2


def _f32(v):
    return float(np.float32(v))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def philox4x32_10(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_ptr(ctr), _ptr(key), _ptr(out))
    return out


def active(seed, step, replica, skip_prob, delay_replica=0, delay_rounds=0):
    return int(lib().oracle_active_ex(seed, step, replica, skip_prob, delay_replica, delay_rounds))


def peer(seed, step, layer, replica, K, peer_mode=0):
    return int(lib().oracle_peer(seed, step, layer, replica, K, peer_mode))


def schedule(seed, step, L, K, peer_mode=0, skip_prob=0.0, delay_replica=0, delay_rounds=0):
    """-> (peer[L,K] int32 with -1 for inactive replicas, active[K] uint8)."""
    p = np.empty((L, K), dtype=np.int32)
    a = np.empty(K, dtype=np.uint8)
    lib().oracle_schedule(seed, step, L, K, peer_mode, skip_prob, delay_replica, delay_rounds, _ptr(p), _ptr(a))
    return p, a


def mix_tables(w, peer, active, mix_mode=0):
    """-> (recv_off[K+1], senders[n], alpha[n], w_new[K]) for one (step, layer): the sender list of
    every receiver in ascending order with the coefficient of each push (oracle_mix_tables)."""
    w = np.ascontiguousarray(w, dtype=np.float64)
    K = w.shape[0]
    peer = np.ascontiguousarray(peer, dtype=np.int32)
    active = np.ascontiguousarray(active, dtype=np.uint8)
    recv_off = np.zeros(K + 1, dtype=np.int32)
    senders = np.zeros(K, dtype=np.int32)
    alpha = np.zeros(K, dtype=np.float32)
    w_new = np.empty(K, dtype=np.float64)
    lib().oracle_mix_tables(K, _ptr(w), _ptr(peer), _ptr(active), mix_mode, _ptr(recv_off), _ptr(senders), _ptr(alpha),
                            _ptr(w_new))
    n = int(recv_off[K])
    return recv_off, senders[:n].copy(), alpha[:n].copy(), w_new


def disagreement(x, w=None):
    """dist[i] = ||x_i - xbar||^2 over one layer; x: [K, n] fp32; w: [K] fp64 weights or None (plain mean)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    K, n = x.shape
    if w is not None:
        w = np.ascontiguousarray(w, dtype=np.float64)
    out = np.empty(K, dtype=np.float64)
    lib().oracle_disagreement(K, n, _ptr(x), _ptr(w), _ptr(out))
    return out


def layer_update(x, g, m, w, lr, mu, seed, step, layer, peer_mode=0, skip_prob=0.0,
                 peer_in=None, active_in=None, delay_replica=0, delay_rounds=0):
    """One (step, layer) in place.  x, g, m: [K, n] (fp32, or x/m fp64 for the shadow); w: [K] fp64."""
    K, n = x.shape
    f64 = x.dtype == np.float64
    assert x.flags.c_contiguous and g.flags.c_contiguous and w.flags.c_contiguous
    assert g.dtype == np.float32 and g.shape == x.shape and w.dtype == np.float64 and w.shape == (K,)
    if mu != 0.0:
        assert m is not None and m.dtype == x.dtype and m.shape == x.shape and m.flags.c_contiguous
    if peer_in is not None:
        peer_in = np.ascontiguousarray(peer_in, dtype=np.int32)
    if active_in is not None:
        active_in = np.ascontiguousarray(active_in, dtype=np.uint8)
    f = lib().oracle_layer_update_f64 if f64 else lib().oracle_layer_update
    rc = f(K, n, _ptr(x), _ptr(g), _ptr(m) if mu != 0.0 else None, _ptr(w), lr, mu, seed, step, layer,
           peer_mode, skip_prob, delay_replica, delay_rounds, _ptr(peer_in), _ptr(active_in))
    if rc != 0:
        raise MemoryError("oracle_layer_update failed")


def layer_update_ex(x, g, m, v, w, bpow, tcount, lr, mu=0.0, wd=0.0, beta1=0.9, beta2=0.999, eps=1e-8,
                    optimizer=OPT_SGD, mix_mode=MIX_PUSHSUM, seed=0, step=0, layer=0, peer_mode=0, skip_prob=0.0,
                    peer_in=None, active_in=None, delay_replica=0, delay_rounds=0):
    """One (step, layer) of the widened rule (NEXT-3 optimisers, NEXT-4 mixers) in place.
    x, m, v: [K, n] fp32 (or fp64 for the shadow); g: [K, n] fp32; w: [K] fp64;
    bpow: [K, 2] fp64 and tcount: [K] int64 (AdamW only, else None)."""
    K, n = x.shape
    f64 = x.dtype == np.float64
    assert x.flags.c_contiguous and g.flags.c_contiguous and w.flags.c_contiguous
    assert g.dtype == np.float32 and g.shape == x.shape and w.dtype == np.float64 and w.shape == (K,)
    need_m = optimizer == OPT_ADAMW or mu != 0.0
    for a, need in ((m, need_m), (v, optimizer == OPT_ADAMW)):
        if need:
            assert a is not None and a.dtype == x.dtype and a.shape == x.shape and a.flags.c_contiguous
    if optimizer == OPT_ADAMW:
        assert bpow.dtype == np.float64 and bpow.shape == (K, 2) and bpow.flags.c_contiguous
        assert tcount.dtype == np.int64 and tcount.shape == (K,)
    if peer_in is not None:
        peer_in = np.ascontiguousarray(peer_in, dtype=np.int32)
    if active_in is not None:
        active_in = np.ascontiguousarray(active_in, dtype=np.uint8)
    o = _Opts(optimizer, mix_mode, _f32(lr), _f32(mu), _f32(wd), _f32(beta1), _f32(beta2), _f32(eps))
    f = lib().oracle_layer_update_ex_f64 if f64 else lib().oracle_layer_update_ex
    rc = f(K, n, _ptr(x), _ptr(g), _ptr(m) if need_m else None, _ptr(v) if optimizer == OPT_ADAMW else None, _ptr(w),
           _ptr(bpow) if optimizer == OPT_ADAMW else None, _ptr(tcount) if optimizer == OPT_ADAMW else None,
           ctypes.byref(o), seed, step, layer, peer_mode, skip_prob, delay_replica, delay_rounds,
           _ptr(peer_in), _ptr(active_in))
    if rc != 0:
        raise MemoryError("oracle_layer_update_ex failed")


class Oracle:
    """State of K replicas of L layers; round(step, grads) walks the layers L-1 .. 0
    (output layer first)."""

    def __init__(self, numel, K, lr, momentum=0.0, seed=0, peer_mode=0, skip_prob=0.0, f64=False,
                 delay_replica=0, delay_rounds=0, optimizer=OPT_SGD, mix_mode=MIX_PUSHSUM, weight_decay=0.0,
                 beta1=0.9, beta2=0.999, eps=1e-8):
        self.numel = [int(n) for n in numel]
        self.L, self.K = len(self.numel), int(K)
        self.lr, self.mu = lr, momentum
        self.seed, self.peer_mode, self.skip_prob = int(seed), int(peer_mode), float(skip_prob)
        self.delay_replica, self.delay_rounds = int(delay_replica), int(delay_rounds)
        self.dt = np.float64 if f64 else np.float32
        self.x = [np.zeros((self.K, n), dtype=self.dt) for n in self.numel]
        self.optimizer, self.mix_mode, self.wd = int(optimizer), int(mix_mode), float(weight_decay)
        self.beta1, self.beta2, self.eps = float(beta1), float(beta2), float(eps)
        adam = self.optimizer == OPT_ADAMW
        self.m = [np.zeros((self.K, n), dtype=self.dt) for n in self.numel] if (momentum != 0.0 or adam) else None
        self.v = [np.zeros((self.K, n), dtype=self.dt) for n in self.numel] if adam else None
        self.bpow = np.ones((self.L, self.K, 2), dtype=np.float64) if adam else None
        self.tcount = np.zeros((self.L, self.K), dtype=np.int64) if adam else None
        self.w = np.full((self.L, self.K), 1.0 / self.K, dtype=np.float64)

    def layer_update(self, step, layer, g):
        g = np.ascontiguousarray(g, dtype=np.float32)
        if self.optimizer == OPT_SGD and self.mix_mode == MIX_PUSHSUM and self.wd == 0.0:
            lr = float(np.float32(self.lr)) if self.dt == np.float64 else self.lr
            mu = float(np.float32(self.mu)) if self.dt == np.float64 else self.mu
            layer_update(self.x[layer], g, self.m[layer] if self.m is not None else None, self.w[layer],
                         lr, mu, self.seed, step, layer, self.peer_mode, self.skip_prob,
                         delay_replica=self.delay_replica, delay_rounds=self.delay_rounds)
            return
        adam = self.optimizer == OPT_ADAMW
        layer_update_ex(self.x[layer], g, self.m[layer] if self.m is not None else None,
                        self.v[layer] if adam else None, self.w[layer],
                        self.bpow[layer] if adam else None, self.tcount[layer] if adam else None,
                        self.lr, self.mu, self.wd, self.beta1, self.beta2, self.eps, self.optimizer, self.mix_mode,
                        self.seed, step, layer, self.peer_mode, self.skip_prob,
                        delay_replica=self.delay_replica, delay_rounds=self.delay_rounds)

    def disagreement(self, weighted=False):
        """[L, K] squared distances to the (weighted) consensus, per layer."""
        return np.stack([disagreement(np.asarray(self.x[l], dtype=np.float32), self.w[l] if weighted else None)
                         for l in range(self.L)])

    def round(self, step, grads):
        for layer in reversed(range(self.L)):
            self.layer_update(step, layer, grads[layer])
