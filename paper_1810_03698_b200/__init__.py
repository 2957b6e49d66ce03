"""B200-native treecode-BEM Poisson-Boltzmann hot path (arXiv:1810.03698).

`paper_1810_03698_b200.pb` is the thin binding over the C-ABI library
(include/pb.h); `paper_1810_03698_b200.workloads` draws the seeded synthetic inputs.
Importing this package loads neither; `pb` fails loudly if the CUDA library is absent.
"""
