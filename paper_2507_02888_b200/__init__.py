"""B200-native batched Ewald summation (arxiv 2507.02888 hot path).  See DESIGN.md.

The CUDA library is loaded lazily on first use (paper_2507_02888_b200.ewald); importing the package
or its seeded input generators (paper_2507_02888_b200.workloads) needs no GPU.
"""
