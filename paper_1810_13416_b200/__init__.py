"""B200-native PPM+PPB timestep (arxiv/paper_1810_13416 hot path).  See DESIGN.md.

`workloads` (seeded synthetic inputs) is importable without the CUDA library; everything in
`binding` loads the in-tree C-ABI library and fails loudly if it is missing.
"""
