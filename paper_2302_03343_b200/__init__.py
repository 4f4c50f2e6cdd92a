"""B200-native (sm_100a) batched PDF interpolation: the hot path of PDFFlow
(M. Rossi, arXiv:2302.03343, ch. 3-4) behind a C ABI (include/pdfgrid.h).

``paper_2302_03343_b200.synth``   seeded synthetic workloads (no method arithmetic)
``paper_2302_03343_b200.binding`` thin ctypes binding of libpdfgrid.so (loaded lazily;
                                  raises if the CUDA library is missing - no CPU fallback)
"""
__all__ = ["synth", "binding", "shard"]
