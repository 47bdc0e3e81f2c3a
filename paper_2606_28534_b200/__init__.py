"""B200-native BIT1-style 1D3V PIC-MC hot path (arxiv/paper_2606_28534).

`workloads` (seeded input generators) imports without a GPU; `binding` loads the
C-ABI CUDA library (libbit1.so) lazily and fails loudly when it is missing.
"""
