"""paper_1411_0436_b200 — B200-native (sm_100a) streaming spectrometer hot path of arXiv 1411.0436.

unpack int8 -> polyphase FIR -> N-point FFT -> Stokes products -> fp32 accumulate, all in
hand-written CUDA behind the C-ABI library declared in include/spec.h.  This package holds the
CUDA sources (csrc/), the build step (build.py), the ctypes binding (spec.py: argument
marshalling only) and the seeded input generators (synth.py).  Importing the package does not
load the CUDA library; `spec` does, and fails loudly if it is missing.
"""
__all__ = ["spec", "synth", "build"]
