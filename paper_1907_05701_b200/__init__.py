"""paper_1907_05701_b200 -- B200-native super-learner step of Hierarchical ADPSGD.

The product is libhadpsgd.so (hand-written sm_100a CUDA behind the C ABI of
include/hadpsgd.h); this package is its thin Python binding.  No CPU fallback.
"""
from .binding import (BF16, DETERMINISTIC, EQ7_LITERAL, F32, NO_DIAG, NO_MIX, PEER, SHARE_PAIR_WEIGHTS, Hadpsgd,  # noqa: F401
                      HadpsgdError, hadpsgd_consensus_noalloc, hadpsgd_plan_peer, hadpsgd_plan_slots,
                      hadpsgd_layout, hadpsgd_lr_schedule, hadpsgd_pairing, hadpsgd_required_bytes,
                      hadpsgd_shard_range, lib)
