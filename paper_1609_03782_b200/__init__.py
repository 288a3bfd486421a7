"""B200-native intensity-driven gradient (IDG) filter, arXiv:1609.03782 section 3.3.

The product is the C-ABI library built from ``csrc/`` (declared in ``include/idg.h``);
``binding`` marshals torch CUDA tensors into it.  Nothing here falls back to the CPU.
"""
__version__ = "0.1.0"
