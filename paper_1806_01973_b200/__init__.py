"""paper_1806_01973_b200 -- B200-native (sm_100a) PinSage layer-wise inference.

The product is the C-ABI library built from ``csrc/`` (``include/pinsage.h``);
``binding`` is its thin ctypes front-end and ``synth`` the seeded input generators.
Importing the package does not load the CUDA library; the first call through
``binding`` does, and fails loudly if it is missing (there is no CPU fallback).
"""
__version__ = "0.1.0"
