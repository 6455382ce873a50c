"""B200-native explicit OSB-PD time stepper (arXiv 2309.11273 hot path).

`paper_2309_11273_b200.pd` is the thin binding over the C-ABI library (csrc/ -> libpd.so);
`paper_2309_11273_b200.workloads` holds the seeded synthetic input generators and imports
neither the binding nor the oracle.  Nothing here falls back to a CPU path: using the
binding without the built CUDA library raises.
"""
__all__ = ["pd", "workloads"]
