"""Energy-test hot path (arXiv:1612.04705) for NVIDIA B200 (sm_100a).

The product is the C-ABI library ``libet.so`` (``include/et.h``) built from
``csrc/``; ``binding`` is its thin ctypes front and ``datagen`` the seeded
synthetic inputs.  Importing the package does not load the CUDA library;
``binding.lib()`` does, and fails loudly when it is missing.
"""
__all__ = ["binding", "datagen", "build"]
