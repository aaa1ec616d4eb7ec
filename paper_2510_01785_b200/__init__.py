"""B200-native HEALPix spherical harmonic transforms (cuHPX hot path, arXiv 2510.01785)."""
