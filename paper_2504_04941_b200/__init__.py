"""B200-native per-cell implicit thermochemistry step (arxiv 2504.04941, sections 2.2-2.3).

``workloads`` (numpy only) draws the seeded synthetic inputs; ``binding`` is the
thin ctypes layer over the C-ABI library ``libkratos_chem.so`` built from ``csrc/``.
Nothing here falls back to the CPU: without the CUDA library the calls raise.
"""
__all__ = ["workloads", "binding"]
