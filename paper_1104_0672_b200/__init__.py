"""arkcos-b200: B200-native (sm_100a) hybrid ring convolution on the sphere (arXiv:1104.0672).

The product is the C-ABI library ``libarkcos.so`` (include/arkcos.h); ``arkcos`` is the thin ctypes
binding with the same names; ``inputs`` holds the seeded synthetic inputs.  Importing this package
loads nothing native; the binding loads the library on first use and fails loudly if it is missing.
"""
__all__ = ["arkcos", "inputs"]
