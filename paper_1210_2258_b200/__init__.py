"""paper_1210_2258_b200 -- B200-native SGP / Richardson-Lucy deconvolution (arXiv:1210.2258).

The product is the C-ABI CUDA library `libsgp_b200.so` (include/sgp.h); `binding` holds the thin
ctypes layer with the same entry-point names, `synth` the seeded synthetic workloads.
Nothing here imports the CPU oracle.
"""
__version__ = "0.1.0"
