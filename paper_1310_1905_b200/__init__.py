"""paper_1310_1905_b200: the super-droplet (particle-based) warm-rain step of arxiv 1310.1905 on one B200.

``binding``   ctypes binding of the C-ABI library libsdm.so (include/sdm.h), built from ``csrc/``.
``workloads`` seeded synthetic inputs (the box, 2D and 3D set-ups of BASELINE.json).
``build``     nvcc build of libsdm.so for sm_100a.
Nothing here imports ``oracle``.
"""
__all__ = ["binding", "workloads", "build"]
