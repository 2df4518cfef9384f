"""B200-native QC-LDPC syndrome belief-propagation decoder (hot path of arXiv 1702.07740).

`workloads` (seeded synthetic inputs) imports without the CUDA extension; everything in `binding` needs
`csrc/libqcldpc.so` and fails loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "binding"]
