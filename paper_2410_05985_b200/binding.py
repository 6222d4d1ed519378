"""ctypes binding of include/layup.h -- argument marshalling only.

Every step of the path runs in the kernels of csrc/*.cu.  torch is used for device
memory (the arena is a torch uint8 tensor) and streams; nothing here computes.  If
csrc/liblayup.so is missing or no CUDA device is present, calls fail loudly.
"""
import ctypes
import os
from typing import List, Optional, Sequence

import numpy as np
import torch

LAYUP_OK, LAYUP_EINVAL, LAYUP_ESTATE, LAYUP_ECUDA = 0, -1, -2, -3
WHAT_X, WHAT_G, WHAT_M, WHAT_V = 0, 1, 2, 3
OPT_SGD, OPT_ADAMW = 0, 1
MIX_PUSHSUM, MIX_LOSSY, MIX_SYMMETRIC = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "csrc", "liblayup.so")
_lib = None


class LayUpError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("layup error %d: %s" % (code, text))
        self.code = code


class _Tuning(ctypes.Structure):
    """layup_tuning of include/layup.h: 0 = the library's default in every field."""
    _fields_ = [(n, ctypes.c_int32) for n in ("engine", "launch_shape", "fused", "fused_waves", "tile_items", "variant",
                                              "ctas_per_sm", "pdl", "tma2d", "stages", "group_threads")]


ENGINE_TMA, ENGINE_LDG = 1, 2
SHAPE_GROUPED, SHAPE_PERSISTENT = 1, 2
FUSED_AUTO, FUSED_NEVER = 1, 2


class _Config(ctypes.Structure):
    _fields_ = [("K", ctypes.c_int32), ("L", ctypes.c_int32), ("numel", ctypes.POINTER(ctypes.c_int64)),
                ("lr", ctypes.c_float), ("momentum", ctypes.c_float), ("seed", ctypes.c_uint64),
                ("peer_mode", ctypes.c_int32), ("skip_prob", ctypes.c_float), ("device", ctypes.c_int32),
                ("delay_replica", ctypes.c_int32), ("delay_rounds", ctypes.c_int32),
                ("optimizer", ctypes.c_int32), ("mix_mode", ctypes.c_int32), ("weight_decay", ctypes.c_float),
                ("beta1", ctypes.c_float), ("beta2", ctypes.c_float), ("eps", ctypes.c_float),
                ("tuning", ctypes.POINTER(_Tuning))]


EXPORTS = ["layup_arena_bytes", "layup_init", "layup_destroy", "layup_ptr", "layup_set_lr",
           "layup_layer_update", "layup_round", "layup_round_host", "layup_sync", "layup_peer",
           "layup_schedule", "layup_schedule_tables", "layup_last_order", "layup_trace", "layup_trace_read",
           "layup_weights", "layup_state_export", "layup_state_import", "layup_disagreement", "layup_disagreement_ms",
           "layup_disagreement_static",
           "layup_graph_begin", "layup_graph_end", "layup_graph_launch", "layup_graph_destroy",
           "layup_profile", "layup_profile_read", "layup_launch_count", "layup_last_error"]


def load_library():
    """dlopen csrc/liblayup.so (built by __graft_entry__.build()); no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise LayUpError(LAYUP_ECUDA, "%s not built: run `python -c 'import __graft_entry__ as g; g.build()'`" % _SO)
    lib = ctypes.CDLL(_SO)
    c = ctypes
    vp, i32, i64 = c.c_void_p, c.c_int32, c.c_int64
    sig = {
        "layup_arena_bytes": [c.POINTER(_Config), c.POINTER(c.c_size_t)],
        "layup_init": [c.POINTER(_Config), vp, c.c_size_t, c.POINTER(vp)],
        "layup_destroy": [vp],
        "layup_ptr": [vp, i32, i32, i32, c.POINTER(vp), c.POINTER(i64)],
        "layup_set_lr": [vp, c.c_float],
        "layup_layer_update": [vp, i64, i32, vp],
        "layup_round": [vp, i64, vp],
        "layup_round_host": [vp, i64, vp, vp],
        "layup_sync": [vp],
        "layup_peer": [c.c_uint64, i64, i32, i32, i32, c.POINTER(i32)],
        "layup_schedule": [vp, i64, vp, vp],
        "layup_weights": [vp, vp],
        "layup_state_export": [vp, vp, vp, vp],
        "layup_state_import": [vp, vp, vp, vp],
        "layup_disagreement": [vp, i32, vp, vp],
        "layup_disagreement_ms": [vp, c.POINTER(c.c_double)],
        "layup_disagreement_static": [vp, i32, i32, c.POINTER(i64), vp, vp, vp],
        "layup_schedule_tables": [vp, i32, c.POINTER(i64), vp, vp, vp, vp, vp],
        "layup_last_order": [vp, vp, c.POINTER(i32)],
        "layup_trace": [vp, i32],
        "layup_trace_read": [vp, vp],
        "layup_graph_begin": [vp, vp],
        "layup_graph_end": [vp, c.POINTER(vp)],
        "layup_graph_launch": [vp, vp, vp],
        "layup_graph_destroy": [vp, vp],
        "layup_profile": [vp, i32],
        "layup_profile_read": [vp, c.POINTER(i64), c.POINTER(c.c_double)],
        "layup_launch_count": [vp, c.POINTER(i64)],
    }
    for name, args in sig.items():
        f = getattr(lib, name)
        f.argtypes, f.restype = args, c.c_int
    lib.layup_last_error.argtypes, lib.layup_last_error.restype = [vp], c.c_char_p
    _lib = lib
    return lib


def _check(rc, ctx=None):
    if rc != LAYUP_OK:
        raise LayUpError(rc, (load_library().layup_last_error(ctx) or b"").decode())


def _config(K, numel, lr, momentum, seed, peer_mode, skip_prob, device, delay_replica=0, delay_rounds=0,
            optimizer=OPT_SGD, mix_mode=MIX_PUSHSUM, weight_decay=0.0, beta1=0.9, beta2=0.999, eps=1e-8, tuning=None):
    arr = (ctypes.c_int64 * len(numel))(*[int(n) for n in numel])
    tune = _Tuning(**{k: int(v) for k, v in tuning.items()}) if tuning else None
    cfg = _Config(int(K), len(numel), arr, float(lr), float(momentum), int(seed), int(peer_mode),
                  float(skip_prob), int(device), int(delay_replica), int(delay_rounds),
                  int(optimizer), int(mix_mode), float(weight_decay), float(beta1), float(beta2), float(eps),
                  ctypes.pointer(tune) if tune is not None else None)
    cfg._keep = (arr, tune)
    return cfg


def layup_arena_bytes(K, numel, momentum=0.0, optimizer=OPT_SGD) -> int:
    out = ctypes.c_size_t(0)
    cfg = _config(K, numel, 0.0, momentum, 0, 0, 0.0, 0, optimizer=optimizer)
    _check(load_library().layup_arena_bytes(ctypes.byref(cfg), ctypes.byref(out)))
    return out.value


def layup_peer(seed, step, layer, replica, K) -> int:
    out = ctypes.c_int32(0)
    _check(load_library().layup_peer(int(seed), int(step), int(layer), int(replica), int(K), ctypes.byref(out)))
    return out.value


_raw_stream = getattr(torch._C, "_cuda_getCurrentRawStream", None)


def _stream_handle(stream, device_index=None) -> Optional[int]:
    if stream is None:
        if _raw_stream is not None and device_index is not None:
            return _raw_stream(device_index) or None
        return torch.cuda.current_stream().cuda_stream or None
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream or None
    return int(stream) or None


def layup_disagreement_static(x_dev, K: int, numel: Sequence[int], w: Optional[np.ndarray] = None,
                              stream=None) -> np.ndarray:
    """layup_disagreement for callers that must not allocate device memory (include/layup.h): no ctx,
    no cudaMalloc -- the kernel's accumulators sit in an array compiled into liblayup.so, which caps
    len(numel) * K at LAYUP_STATIC_MAX_PAIRS.  Meant for a monitoring hook that runs while backward and
    gossip overlap (a cudaMalloc there stalls the whole device) or for a process that only borrows an
    X section and has no ctx.  x_dev: raw device address (int) of an X section in the arena layout on the
    CURRENT device, e.g. LayUp.ptr(WHAT_X, 0, 0)[0]; w: [L, K] float64 consensus coefficients or None
    for the plain mean.  Returns dist[L, K].  Synchronous; concurrent callers are serialised by the
    library because they all share that one array."""
    L = len(numel)
    arr = (ctypes.c_int64 * L)(*[int(v) for v in numel])
    wd = None if w is None else np.ascontiguousarray(w, dtype=np.float64).reshape(L, int(K))
    d = np.empty((L, int(K)), dtype=np.float64)
    sh = _stream_handle(stream, torch.cuda.current_device()) if torch.cuda.is_available() else None
    _check(load_library().layup_disagreement_static(int(x_dev), int(K), L, arr, None if wd is None else wd.ctypes.data,
                                                    d.ctypes.data, sh))
    return d


LAYUP_STATIC_MAX_PAIRS = 16384


class LayUp:
    """One ctx = K replicas of L layers in one torch-allocated arena on one GPU."""

    def __init__(self, K: int, numel: Sequence[int], lr: float, momentum: float = 0.0, seed: int = 0,
                 peer_mode: int = 0, skip_prob: float = 0.0, device: int = 0,
                 delay_replica: int = 0, delay_rounds: int = 0, optimizer: int = OPT_SGD,
                 mix_mode: int = MIX_PUSHSUM, weight_decay: float = 0.0, beta1: float = 0.9, beta2: float = 0.999,
                 eps: float = 1e-8, tuning: Optional[dict] = None):
        """tuning: layup_tuning fields by name (include/layup.h), e.g. dict(launch_shape=SHAPE_PERSISTENT)."""
        self.lib = load_library()
        self.K, self.L, self.numel = int(K), len(numel), [int(n) for n in numel]
        self.momentum = float(momentum)
        self.device = torch.device("cuda", device)
        self.optimizer, self.mix_mode = int(optimizer), int(mix_mode)
        self._cfg = _config(K, numel, lr, momentum, seed, peer_mode, skip_prob, device, delay_replica, delay_rounds,
                            optimizer, mix_mode, weight_decay, beta1, beta2, eps, tuning)
        nbytes = ctypes.c_size_t(0)
        _check(self.lib.layup_arena_bytes(ctypes.byref(self._cfg), ctypes.byref(nbytes)))
        self.arena_bytes = nbytes.value
        if not torch.cuda.is_available():
            raise LayUpError(LAYUP_ECUDA, "no CUDA device: the LayUp path has no CPU fallback")
        self.arena = torch.empty(self.arena_bytes + 128, dtype=torch.uint8, device=self.device)
        shift = (-self.arena.data_ptr()) % 128
        self._arena_f32 = self.arena[shift:shift + self.arena_bytes].view(torch.float32)
        torch.cuda.synchronize(self.device)
        ctx = ctypes.c_void_p()
        _check(self.lib.layup_init(ctypes.byref(self._cfg), self._arena_f32.data_ptr(), self.arena_bytes,
                                   ctypes.byref(ctx)))
        self.ctx = ctx
        self._base = self._arena_f32.data_ptr()

    # -- arena views (torch plumbing: a view is a slice of the arena tensor) --------------
    def ptr(self, what: int, replica: int, layer: int):
        p, n = ctypes.c_void_p(), ctypes.c_int64()
        _check(self.lib.layup_ptr(self.ctx, what, replica, layer, ctypes.byref(p), ctypes.byref(n)), self.ctx)
        return p.value, n.value

    def view(self, what: int, layer: int) -> torch.Tensor:
        """[K, numel] fp32 strided view of all replicas of one layer."""
        p0, n = self.ptr(what, 0, layer)
        off0 = (p0 - self._base) // 4
        if self.K > 1:
            p1, _ = self.ptr(what, 1, layer)
            stride = (p1 - p0) // 4
        else:
            stride = (n + 31) // 32 * 32
        return self._arena_f32.as_strided((self.K, n), (stride, 1), off0)

    # -- the C-ABI calls, same names -----------------------------------------------------
    def layup_set_lr(self, lr: float):
        _check(self.lib.layup_set_lr(self.ctx, lr), self.ctx)

    def layup_layer_update(self, step: int, layer: int, stream=None):
        _check(self.lib.layup_layer_update(self.ctx, step, layer, _stream_handle(stream, self.device.index)), self.ctx)

    def layup_round(self, step: int, stream=None):
        _check(self.lib.layup_round(self.ctx, step, _stream_handle(stream, self.device.index)), self.ctx)

    def layup_round_host(self, step: int, g_host: torch.Tensor, x_host: Optional[torch.Tensor]):
        _check(self.lib.layup_round_host(self.ctx, step, g_host.data_ptr(),
                                         x_host.data_ptr() if x_host is not None else None), self.ctx)

    def layup_sync(self):
        _check(self.lib.layup_sync(self.ctx), self.ctx)

    def layup_schedule(self, step: int):
        peer = np.empty((self.L, self.K), dtype=np.int32)
        active = np.empty(self.K, dtype=np.uint8)
        _check(self.lib.layup_schedule(self.ctx, step, peer.ctypes.data, active.ctypes.data), self.ctx)
        return peer, active

    def layup_schedule_tables(self, layer: int):
        """-> dict(step, peer[K], flags[K], recv_off[K+1], senders[K], alpha[K]) as the update kernel consumed them."""
        K = self.K
        step = ctypes.c_int64()
        peer, flags = np.empty(K, dtype=np.int32), np.empty(K, dtype=np.uint8)
        recv_off, senders = np.empty(K + 1, dtype=np.int32), np.empty(K, dtype=np.int32)
        alpha = np.empty(K, dtype=np.float32)
        _check(self.lib.layup_schedule_tables(self.ctx, layer, ctypes.byref(step), peer.ctypes.data, flags.ctypes.data,
                                              recv_off.ctypes.data, senders.ctypes.data, alpha.ctypes.data), self.ctx)
        return dict(step=step.value, peer=peer, flags=flags, recv_off=recv_off, senders=senders, alpha=alpha)

    def layup_last_order(self) -> List[int]:
        out, n = np.empty(self.L, dtype=np.int32), ctypes.c_int32()
        _check(self.lib.layup_last_order(self.ctx, out.ctypes.data, ctypes.byref(n)), self.ctx)
        return [int(v) for v in out[:n.value]]

    def layup_trace(self, enable: bool):
        _check(self.lib.layup_trace(self.ctx, 1 if enable else 0), self.ctx)

    def layup_trace_read(self) -> np.ndarray:
        out = np.empty(self.L, dtype=np.uint64)
        _check(self.lib.layup_trace_read(self.ctx, out.ctypes.data), self.ctx)
        return out

    def layup_graph_begin(self, stream):
        _check(self.lib.layup_graph_begin(self.ctx, _stream_handle(stream, self.device.index)), self.ctx)

    def layup_graph_end(self):
        g = ctypes.c_void_p()
        _check(self.lib.layup_graph_end(self.ctx, ctypes.byref(g)), self.ctx)
        return g

    def layup_graph_launch(self, graph, stream=None):
        _check(self.lib.layup_graph_launch(self.ctx, graph, _stream_handle(stream, self.device.index)), self.ctx)

    def layup_graph_destroy(self, graph):
        _check(self.lib.layup_graph_destroy(self.ctx, graph), self.ctx)

    def layup_weights(self) -> np.ndarray:
        w = np.empty((self.L, self.K), dtype=np.float64)
        _check(self.lib.layup_weights(self.ctx, w.ctypes.data), self.ctx)
        return w

    def layup_state_export(self):
        """-> (w [L,K] fp64, bpow [L,K,2] fp64 or None, next_step [L] int64)."""
        w = np.empty((self.L, self.K), dtype=np.float64)
        bp = np.empty((self.L, self.K, 2), dtype=np.float64) if self.optimizer == OPT_ADAMW else None
        ns = np.empty(self.L, dtype=np.int64)
        _check(self.lib.layup_state_export(self.ctx, w.ctypes.data, bp.ctypes.data if bp is not None else None,
                                           ns.ctypes.data), self.ctx)
        return w, bp, ns

    def layup_state_import(self, w, bpow, next_step):
        w = np.ascontiguousarray(w, dtype=np.float64)
        ns = np.ascontiguousarray(next_step, dtype=np.int64)
        bp = np.ascontiguousarray(bpow, dtype=np.float64) if bpow is not None else None
        assert w.shape == (self.L, self.K) and ns.shape == (self.L,)
        _check(self.lib.layup_state_import(self.ctx, w.ctypes.data, bp.ctypes.data if bp is not None else None,
                                           ns.ctypes.data), self.ctx)

    def layup_disagreement(self, weighted: bool = False, stream=None) -> np.ndarray:
        d = np.empty((self.L, self.K), dtype=np.float64)
        _check(self.lib.layup_disagreement(self.ctx, 1 if weighted else 0, d.ctypes.data,
                                           _stream_handle(stream, self.device.index)), self.ctx)
        return d

    def layup_disagreement_ms(self) -> float:
        ms = ctypes.c_double()
        _check(self.lib.layup_disagreement_ms(self.ctx, ctypes.byref(ms)), self.ctx)
        return ms.value

    def layup_profile(self, enable: bool):
        _check(self.lib.layup_profile(self.ctx, 1 if enable else 0), self.ctx)

    def layup_profile_read(self):
        n, ms = ctypes.c_int64(), ctypes.c_double()
        _check(self.lib.layup_profile_read(self.ctx, ctypes.byref(n), ctypes.byref(ms)), self.ctx)
        return n.value, ms.value

    def layup_launch_count(self) -> int:
        n = ctypes.c_int64()
        _check(self.lib.layup_launch_count(self.ctx, ctypes.byref(n)), self.ctx)
        return n.value

    def close(self):
        if getattr(self, "ctx", None):
            self.lib.layup_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
