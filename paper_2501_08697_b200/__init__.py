"""B200-native plane-wave Kohn-Sham H*psi and block-Davidson (arxiv 2501.08697, §III.A-B).

`inputs` is importable without the CUDA extension; `kspw` (the binding of libkspw.so) raises
loudly when the library is missing -- there is no CPU fallback.
"""
