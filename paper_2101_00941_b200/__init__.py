"""B200-native streamed dedispersion + single-pulse search (arXiv 2101.00941 hot path).

`paper_2101_00941_b200.binding` is the thin ctypes layer over the C-ABI library
(`include/aa.h`, built from `csrc/`); `paper_2101_00941_b200.inputs` is the
seeded input generator shared by tests, bench and the oracle's tests.
Nothing is imported eagerly: the binding fails loudly if libaa.so is missing.
"""
__all__ = ["binding", "inputs"]
