"""B200-native HEALPix spherical harmonic transforms (cuHPX hot path, arXiv 2510.01785).

``binding`` wraps the C-ABI CUDA library ``libcuhpx.so`` (include/cuhpx.h); ``synth`` holds the seeded
synthetic input recipes.  Importing ``binding`` fails loudly when the library has not been built.
"""
