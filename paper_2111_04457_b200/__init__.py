"""paper_2111_04457_b200 — B200-native even-odd Wilson(-clover) Dirac operator + mixed-precision BiCGStab.

`bq` is the thin ctypes binding of the C-ABI library (include/bq.h, csrc/); `inputs` is the seeded
synthetic input generator shared with the tests of the CPU oracle.
"""
