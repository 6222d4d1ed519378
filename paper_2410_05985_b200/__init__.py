"""B200-native LayUp hot path: layer-wise local SGD step fused with push-sum gossip
mixing over K replicas in one HBM arena (arXiv 2410.05985, Algorithm 1 "Updater
Thread").  The product is csrc/liblayup.so (hand-written sm_100a CUDA behind the C-ABI of
include/layup.h); this package is only the thin ctypes binding.  There is no CPU path.
"""
from .binding import (ENGINE_LDG, ENGINE_TMA, FUSED_AUTO, FUSED_NEVER, SHAPE_GROUPED, SHAPE_PERSISTENT,  # noqa: F401
                      LAYUP_ECUDA, LAYUP_EINVAL, LAYUP_ESTATE, LAYUP_OK, MIX_LOSSY, MIX_PUSHSUM,  # noqa: F401
                      MIX_SYMMETRIC, OPT_ADAMW, OPT_SGD, WHAT_G, WHAT_M, WHAT_V, WHAT_X,
                      LAYUP_STATIC_MAX_PAIRS, LayUp, LayUpError, layup_arena_bytes, layup_disagreement_static, layup_peer,
                      load_library)
