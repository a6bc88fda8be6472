"""B200-native hot path of the BITS method (arXiv 1208.3407): place -> sort -> search -> reduce.

``paper_1208_3407_b200.bits`` is the thin binding of the C ABI (include/bits.h);
``paper_1208_3407_b200.workloads`` holds the seeded synthetic input generators;
``paper_1208_3407_b200.build`` compiles csrc/ into libbits_b200.so.
"""
