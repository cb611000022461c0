"""adept-b200: B200-native per-step EM shower transport (arXiv 2209.15445, AdePT).

`paper_2209_15445_b200.adept` is the thin ctypes binding of the C-ABI CUDA library
(`include/adept.h`); `paper_2209_15445_b200.inputs` builds the synthetic inputs.
"""
