"""paper_2001_02835_b200 -- B200-native FFT-CONV star-product for NSPT series (arXiv:2001.02835).

The product is the C-ABI library ``libnspt.so`` (sources in ``csrc/``, header in
``include/nspt.h``).  ``binding`` is a thin ctypes layer with the same names; ``workloads``
holds the seeded synthetic input generators (numpy only); ``parallel`` is the direction split of
the staple over ranks (one process per GPU, ``torch.distributed``).  Importing this package does not
load the CUDA library; ``paper_2001_02835_b200.binding`` does, and fails loudly if it is
missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "binding", "build", "parallel"]
__version__ = "0.4.0"   # nspt_version() returns 400
