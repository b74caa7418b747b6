"""gwstream: B200-native streaming inference for the hot path of arXiv:2108.12430.

Snapshotter -> DeepClean-style conv autoencoder -> Hann overlap-add + subtraction ->
BBH 1-D CNN classifier, behind the C ABI declared in ``include/gwstream.h``.

Importing the package is cheap and loads nothing native.  ``binding`` loads the
CUDA shared library on first use and raises if it is missing: there is no CPU or
library fallback.  ``synth`` holds only seeded input/parameter generators (it is the
one module the oracle's tests and the CUDA path's tests both draw inputs from).
"""

__all__ = ["binding", "build", "synth", "specs"]
