"""B200-native batched fp64 chemical source term of the XODIAC photochemical model
(arxiv 2512.06729): NASA-7 thermo -> k_f -> k_r -> rates -> dn/dt -> Jacobian values.

The compute path is the C-ABI library `libxodiac.so` (hand-written CUDA, sm_100a);
`binding` holds the thin ctypes wrappers with the same names.  `synth` holds the seeded
input generators (no method arithmetic).  Importing the package does not load the
library; the first call that needs it does, and fails loudly if it is missing.
"""
__all__ = ["synth", "binding", "build"]
