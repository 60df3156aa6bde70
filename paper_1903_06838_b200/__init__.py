"""B200-native pixel-detector reduction chain of arxiv 1903.06838 (dark, gain, common mode,
photon finding, charge summing, subpixel centroid, sparse summarization).

`paper_1903_06838_b200.binding` is the thin ctypes layer over the C ABI of include/pdp.h
(libpdp.so, built from csrc/ by `paper_1903_06838_b200.build`); `synth` holds the seeded
synthetic input generator.  Nothing is imported eagerly so that the generator can be used
without the CUDA library.
"""
__all__ = ["binding", "build", "synth"]
