"""B200-native SPH pipeline of arXiv 2110.02621 behind the C-ABI library libsph.

`paper_2110_02621_b200.sph` is the ctypes binding of include/sph.h (argument
marshalling only); `paper_2110_02621_b200.inputs` holds the seeded input generators.
"""
