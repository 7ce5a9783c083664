"""B200-native charge-readout hot path of the pixelated LArTPC simulation of arXiv 2212.09807.

``paper_2212_09807_b200.lartpc`` is the thin binding over the C-ABI library (include/lartpc.h);
``paper_2212_09807_b200.workloads`` holds the seeded synthetic inputs.
"""
