"""B200-native hot path of FREDopt's superiorized feasibility-seeking plan optimization (arxiv 2509.20012).

`paper_2509_20012_b200.fredopt` is the thin ctypes binding onto the C-ABI library (include/fredopt.h);
`paper_2509_20012_b200.plangen` is the seeded synthetic input generator.  Nothing is imported eagerly:
the binding fails loudly if the CUDA library is missing, and there is no CPU fallback.
"""
__all__ = ["fredopt", "plangen"]
