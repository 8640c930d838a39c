"""B200-native batched Jenga rigid-body step (arxiv/paper_2606_28394 hot path).

`workloads` (input generators) imports without the CUDA library; everything in
`binding` loads csrc/libjenga.so on first use and fails loudly if it is missing.
"""
