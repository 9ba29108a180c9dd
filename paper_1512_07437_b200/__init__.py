"""B200-native all-pairs posterior stage of QuickProbs 2 (arxiv 1512.07437, stage I).

Sub-modules
-----------
inputs   seeded synthetic protein families + the synthetic default model (numpy only; no method arithmetic)
qp       thin ctypes binding over the C-ABI library ``libqp.so`` (include/qp.h); fails loudly if it is missing
multi    pair-list sharding across ranks + the one distance-matrix exchange (torch.distributed)

Nothing here imports ``oracle/``; the oracle is test infrastructure.
"""

__all__ = ["inputs", "qp", "multi"]
