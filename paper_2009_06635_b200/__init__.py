"""pdfb200: B200-native batched PDF xf(x,Q^2) and alpha_s(Q^2) interpolation.

Hot path of PDFFlow (arXiv:2009.06635) as hand-written sm_100a CUDA kernels behind the
C-ABI of ``include/pdfb200.h``.  ``binding`` is the thin ctypes layer (argument marshalling
only); ``workloads`` holds the seeded synthetic input generators.  Importing this package
does not load the CUDA library; ``binding.lib()`` does and fails loudly if it is missing.
"""
from .pdf import PDF, mkPDF  # noqa: E402,F401  (the paper's user-facing object; marshalling only)

__all__ = ["binding", "workloads", "build", "PDF", "mkPDF"]
