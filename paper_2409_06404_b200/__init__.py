"""B200-native pointwise thermochemistry and mixture-averaged transport (arXiv 2409.06404 hot path).

``workloads``  seeded synthetic mechanism descriptions and states (shared input generators)
``packer``     host-side mechanism packer: description -> species-major SoA tables
``binding``    thin ctypes binding of the C-ABI library ``libcrf.so`` (include/crf.h)
``build``      nvcc build of ``libcrf.so`` for sm_100a
"""
__all__ = ["workloads", "packer", "binding", "build"]
