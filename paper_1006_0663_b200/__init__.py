"""B200-native hot path of the Teukolsky time-stepper of arXiv:1006.0663 (§III.B).

`paper_1006_0663_b200.teuk`   — thin ctypes binding over the C-ABI library `libteuk.so`
                                 (include/teuk.h); raises at import if the library is missing.
`paper_1006_0663_b200.inputs` — seeded synthetic workloads (no method arithmetic).
"""
