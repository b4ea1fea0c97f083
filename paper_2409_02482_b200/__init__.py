"""B200-native renderer for the k-shell rasterise-and-composite path of Volumetric Surfaces
(arXiv 2409.02482).  `synth` = seeded input generators (numpy only); `binding` = thin ctypes
binding of the C-ABI library (include/vs.h), loaded on first use and failing loudly if absent."""

__all__ = ["synth", "binding"]
