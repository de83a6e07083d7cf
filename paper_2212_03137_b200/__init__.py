"""paper_2212_03137_b200 -- B200-native hot path of Quantum-HP (arXiv 2212.03137): RPMD + adQTB MD step.

Thin ctypes binding of the C ABI in `include/qhp.h` (same function names).  Argument marshalling
only: every step of the path runs in the CUDA kernels of `csrc/` (libqhp.so).  PyTorch supplies
device memory and streams.  There is no CPU fallback: importing `binding` without a built
libqhp.so raises, and every call needs a CUDA device.
"""
from .binding import (QHP_THERMO_ADQTB, QHP_THERMO_NONE, QHP_THERMO_PILE, QhpError, System, lib,
                      lib_path, qhp_dfma_probe, qhp_fft_c2c, qhp_philox_normals, qhp_pibar, qhp_pibar_noalloc,
                      PIBAR_NOALLOC_MAX_N)

__all__ = ["System", "QhpError", "lib", "lib_path", "QHP_THERMO_NONE", "QHP_THERMO_PILE",
           "QHP_THERMO_ADQTB", "qhp_philox_normals", "qhp_fft_c2c", "qhp_dfma_probe", "qhp_pibar",
           "qhp_pibar_noalloc", "PIBAR_NOALLOC_MAX_N"]
