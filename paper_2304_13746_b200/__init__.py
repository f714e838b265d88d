"""idfx-b200: B200-native (sm_100a) RK2 Godunov HD / ideal-MHD step of IDEFIX (arXiv 2304.13746).

`paper_2304_13746_b200.idfx` is the thin ctypes binding over the C-ABI library (include/idfx.h);
`paper_2304_13746_b200.inputs` holds the seeded synthetic input generators.  Importing the package does
not load the CUDA library; the first call through the binding does, and fails loudly if it is missing.
"""
