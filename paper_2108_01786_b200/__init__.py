"""B200-native boundary-integral hot path of arXiv 2108.01786: bie_build / bie_matvec / bie_gmres.

``inputs`` (seeded synthetic geometries) is importable without a GPU; the CUDA binding
(``paper_2108_01786_b200.bie``) loads the C-ABI library lazily and fails loudly if it is missing.
"""
__all__ = ["inputs", "bie"]
