"""B200-native spin-parallel Bloch solver (hot path of KomaMRI, arxiv 2301.02702).

``workloads`` (seeded input generators) is importable without the CUDA extension; everything in
``bloch`` needs ``libbloch_b200.so`` and fails loudly when it is missing.
"""
__all__ = ["workloads", "bloch"]
