"""B200-native LVSA block-sparse attention forward (arxiv/paper_2605_31057).

`inputs` (seeded synthetic workloads) is importable on its own; the CUDA path lives in
`binding` (ctypes over csrc/liblvsa.so) and fails loudly when the library cannot be loaded.
"""
