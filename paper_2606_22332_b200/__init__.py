"""B200-native batched tactile readout (after Tactile Genesis, arxiv/paper_2606_22332).

`workloads` is importable without the CUDA library; everything that computes goes through
`paper_2606_22332_b200.binding`, which loads libts.so (hand-written sm_100a CUDA behind the C ABI
of include/ts.h) and raises if it is missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "binding"]
