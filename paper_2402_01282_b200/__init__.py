"""B200-native fp64 directional wavelet transforms on the sphere and ball (arXiv:2402.01282).

`paper_2402_01282_b200.api` is the thin binding over the C-ABI library (include/s2w.h);
`paper_2402_01282_b200.inputs` holds the seeded synthetic inputs.  Importing this package
does not load the CUDA library; `api` does, and fails loudly if it is missing.
"""
