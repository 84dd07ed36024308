"""paper_1206_0675_b200 -- Fourier-accelerated Landau gauge fixing (arXiv:1206.0675) on NVIDIA B200.

The product is the C-ABI library ``liblgf.so`` (include/lgf.h; CUDA sources under ``csrc/``); this
package holds its build script, a thin ctypes binding with the same entry-point names
(``paper_1206_0675_b200.binding``) and the seeded input generators (``inputs``).  Importing the
package loads nothing; the binding loads the CUDA library on first use and fails loudly if it is
missing -- there is no CPU fallback.
"""

__all__ = ["binding", "build", "inputs", "ensemble", "slab"]
__version__ = "0.1.0"
