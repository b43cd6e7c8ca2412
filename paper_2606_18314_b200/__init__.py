"""B200-native exact 2-NN certificate maintenance (arxiv/paper_2606_18314).

The compute lives in ``csrc/`` (hand-written CUDA for sm_100a behind the C-ABI declared in
``include/kc.h``); :mod:`.binding` marshals torch device tensors into it.  There is no CPU
fallback: calling anything in :mod:`.binding` without the built library raises.
:mod:`.workloads` (seeded synthetic inputs) imports without the library.
"""
__all__ = ["binding", "workloads", "driver"]
