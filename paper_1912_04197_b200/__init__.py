"""B200-native fp64 Barnes-Hut gravity (hot path of arxiv/paper_1912_04197).

`binding` is the thin ctypes layer over the C-ABI library declared in include/bh.h (every step of
the path runs in the CUDA kernels under csrc/); `workloads` draws the seeded synthetic inputs;
`build` compiles the library with nvcc for sm_100a.  There is no CPU fallback: `binding` raises if
the library is missing.
"""
