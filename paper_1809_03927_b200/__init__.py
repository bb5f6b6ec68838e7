"""pbs4d -- B200-native hot path of the 4D proton dose calculator of arxiv 1809.03927 (Pepin et al.).

`binding` is the thin ctypes layer over the C-ABI library libpbs4d.so (include/pbs4d.h); `synth` builds the seeded
synthetic inputs; `build` compiles the CUDA sources in-tree.  Nothing here falls back to the CPU: importing
`binding` without the built library, or creating a context without a CUDA device, raises.
"""
__all__ = ["binding", "synth", "build"]
