"""paper_2203_14906_b200 -- B200-native (sm_100a) order-k DMAS photoacoustic beamforming.

Hot path of arXiv 2203.14906 behind the C-ABI library libpab.so (include/pab.h).
`binding` is the thin ctypes layer (argument marshalling only); `synth` is the
seeded input generator shared by tests, bench and the oracle's tests.
Importing the package does not load the CUDA library; `binding.load()` does and
fails loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["synth", "binding"]
