"""paper_2606_08476_b200 — B200-native (sm_100a) implementation of FlashCP's per-CP-rank hot
path (arxiv/paper_2606_08476): plan -> sharding-aware KV gather -> document-masked causal
attention forward/backward -> LSE merge, behind the C ABI of include/fcp.h.

Python here only marshals arguments into libfcp.so; there is no CPU fallback."""
from .binding import (EXPORTS, LIB_PATH, STRATEGY_ALL_PER_DOC, STRATEGY_HYBRID,  # noqa: F401
                      STRATEGY_PER_SEQ, STRATEGY_WHOLE_DOC, PIECE_FULL, PIECE_LOCAL, PIECE_PREFIX,
                      DQ_KEEP, DQ_NO_OUTPUT, STATIC_WORKSPACE_BYTES, TOO_LARGE, FcpError, Plan, Sched, kv_reduce_finish, merge,
                      version)
from .exchange import KVExchange  # noqa: F401,E402
