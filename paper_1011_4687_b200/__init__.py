"""B200-native electrostatic potential / field for QM/MM quantum Monte Carlo.

Hot path of arxiv 1011.4687 (Eq. 4): V(r_i) = sum_j q_j/|r_i - R_j|
and E = -grad V at the QM electrons' positions, as a C-ABI CUDA library
(``include/qmmm_field.h``) plus this thin ctypes binding.  Importing the package
does not load the CUDA library; ``paper_1011_4687_b200.binding`` does, and fails
loudly when it is missing (there is no CPU fallback).
"""
__version__ = "0.1.0"
